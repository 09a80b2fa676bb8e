// qr_backward.cu -- dL/dF scatter-add:
//     dL/dF[i,:] += sum_{p, s : sel_idx[p,s] = i}  sel_w[p,s] * dL_dmap[p,:]
// The selection is piecewise constant in alpha' and the Gaussians are frozen: no other term exists.
//
// Band kernel (K <= kBwdMaxK): CTA = one 16x4-pixel band (64 pixels), 256 threads.
//   1. the band's selection records are read once (coalesced) into shared memory;
//   2. the distinct selected Gaussians of the band (the band union, ~35 rows at K = 40) are numbered with a
//      shared-memory hash set, and the records are scattered into a dense weight block Wr[pixel][64 union rows];
//   3. warp w owns 8 union rows x all D channels in registers (lane = 4 consecutive channels per 128-channel slab),
//      walks the 64 pixels, loads dL_dmap[p,:] (128-bit coalesced) only if the pixel selected one of its rows and
//      accumulates w * g from registers;
//   4. one vector red.global.add per (union row, 4 channels): global atomics drop from (sum of n_sel) * D to
//      (band union) * D -- a 25x pre-reduction at K = 40.
// Pixel kernel (any K): one warp per pixel, vector atomics per selected row -- the plain statement, used for
// K > kBwdMaxK.
#include "qr_backward.cuh"

namespace qr {

constexpr int kBwdThreads = 256;
constexpr int kBwdPx = 64;        // 16 x 4 pixels per CTA
constexpr int kBwdRows = 64;      // union rows per pass (8 warps x 8 rows)
constexpr int kBwdMaxK = 64;


template <int VW> __device__ __forceinline__ void load_g(const float* src, float (&g)[VW]);
template <> __device__ __forceinline__ void load_g<4>(const float* src, float (&g)[4])
{
    const float4 v = __ldg(reinterpret_cast<const float4*>(src));
    g[0] = v.x; g[1] = v.y; g[2] = v.z; g[3] = v.w;
}
template <> __device__ __forceinline__ void load_g<1>(const float* src, float (&g)[1]) { g[0] = __ldg(src); }

template <int VW> __device__ __forceinline__ void red_add(float* dst, const float (&a)[VW]);
template <> __device__ __forceinline__ void red_add<4>(float* dst, const float (&a)[4])
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst), "f"(a[0]), "f"(a[1]), "f"(a[2]), "f"(a[3])
                 : "memory");
}
template <> __device__ __forceinline__ void red_add<1>(float* dst, const float (&a)[1]) { atomicAdd(dst, a[0]); }


template <int NV, int VW>
__global__ void __launch_bounds__(kBwdThreads, 1) backward_band_kernel(const BackwardParams p, const int hs_max /*pow2*/)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int K = p.K, D = p.D;
    float* Wr = reinterpret_cast<float*>(smem_raw);                     // [64 px][64 rows]
    int32_t* rec_slot = reinterpret_cast<int32_t*>(Wr + kBwdPx * kBwdRows);   // [64][K] id, later union slot
    float* rec_w = reinterpret_cast<float*>(rec_slot + kBwdPx * K);     // [64][K]
    int32_t* nsel_s = reinterpret_cast<int32_t*>(rec_w + kBwdPx * K);   // [64]
    int32_t* hkey = nsel_s + kBwdPx;                                    // [hs_max]
    int32_t* hslot = hkey + hs_max;                                     // [hs_max]
    int32_t* uid = hslot + hs_max;                                          // [64*K] union slot -> Gaussian id
    __shared__ int32_t ucount;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x >> 2, band = blockIdx.x & 3;
    const int tile_x = tile % p.cam.tiles_x, tile_y = tile / p.cam.tiles_x;
    const int x0 = tile_x * kTile, y0 = tile_y * kTile + band * 4;
    if (y0 >= p.cam.height) return;
    const int npx = min(kTile, p.cam.width - x0);

    // ---- 1. records -> shared ----
    if (tid == 0) ucount = 0;
    if (tid < kBwdPx) {
        const int px = x0 + (tid & 15), py = y0 + (tid >> 4);
        nsel_s[tid] = (px < p.cam.width && py < p.cam.height) ? p.n_sel[(int64_t)py * p.cam.width + px] : 0;
    }
    __syncthreads();
    int total = 0;
    for (int i = 0; i < kBwdPx; ++i) total += nsel_s[i];    // broadcast reads; same value in every thread
    if (total == 0) return;                                  // uniform: nothing selected in this band
    int hs = 64;
    while (hs < 2 * total) hs <<= 1;                         // <= hs_max by construction (total <= 64 K)
    for (int i = tid; i < hs; i += kBwdThreads) hkey[i] = -1;
    for (int r = 0; r < 4; ++r) {
        const int py = y0 + r;
        if (py >= p.cam.height) break;
        const int64_t gbase = ((int64_t)py * p.cam.width + x0) * K;
        for (int i = tid; i < npx * K; i += kBwdThreads) {
            rec_slot[r * 16 * K + i] = p.sel_idx[gbase + i];
            rec_w[r * 16 * K + i] = p.sel_w[gbase + i];
        }
    }
    __syncthreads();

    // ---- 2a. insert ids into the hash set ----
    const int hmask = hs - 1;
    for (int i = tid; i < kBwdPx * K; i += kBwdThreads) {
        const int lp = i / K, s = i - lp * K;
        if (s < nsel_s[lp]) {
            const int32_t id = rec_slot[i];
            uint32_t h = hash32((uint32_t)id) & hmask;
            while (true) {
                const int32_t old = atomicCAS(&hkey[h], -1, id);
                if (old == -1 || old == id) break;
                h = (h + 1) & hmask;
            }
        }
    }
    __syncthreads();
    // ---- 2b. number the occupied cells ----
    for (int i = tid; i < hs; i += kBwdThreads) {
        const int32_t id = hkey[i];
        if (id >= 0) {
            const int slot = atomicAdd(&ucount, 1);
            hslot[i] = slot;
            uid[slot] = id;
        }
    }
    __syncthreads();
    // ---- 2c. records: id -> union slot ----
    for (int i = tid; i < kBwdPx * K; i += kBwdThreads) {
        const int lp = i / K, s = i - lp * K;
        if (s < nsel_s[lp]) {
            const int32_t id = rec_slot[i];
            uint32_t h = hash32((uint32_t)id) & hmask;
            while (hkey[h] != id) h = (h + 1) & hmask;
            rec_slot[i] = hslot[h];
        }
    }
    const int U = ucount;
    __syncthreads();

    // ---- 3. passes of 64 union rows ----
    for (int c0 = 0; c0 < U; c0 += kBwdRows) {
        for (int i = tid; i < kBwdPx * kBwdRows; i += kBwdThreads) Wr[i] = 0.0f;
        __syncthreads();
        for (int i = tid; i < kBwdPx * K; i += kBwdThreads) {
            const int lp = i / K, s = i - lp * K;
            if (s < nsel_s[lp]) {
                const int slot = rec_slot[i] - c0;
                if (slot >= 0 && slot < kBwdRows) Wr[lp * kBwdRows + slot] = rec_w[i];
            }
        }
        __syncthreads();

        if (c0 + warp * 8 < U) {     // this warp owns rows c0 + warp*8 .. +7
            float acc[8][NV][VW];
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int j = 0; j < NV; ++j)
#pragma unroll
                    for (int v = 0; v < VW; ++v) acc[r][j][v] = 0.0f;

            for (int lp = 0; lp < kBwdPx; ++lp) {
                const float4 w0 = *reinterpret_cast<const float4*>(Wr + lp * kBwdRows + warp * 8);
                const float4 w1 = *reinterpret_cast<const float4*>(Wr + lp * kBwdRows + warp * 8 + 4);
                const float w[8] = { w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w };
                bool any = false;
#pragma unroll
                for (int r = 0; r < 8; ++r) any |= (w[r] != 0.0f);
                if (!any) continue;          // uniform
                const int px = x0 + (lp & 15), py = y0 + (lp >> 4);
                const float* grow = p.dL_dmap + ((int64_t)py * p.cam.width + px) * D;
                float g[NV][VW];
#pragma unroll
                for (int j = 0; j < NV; ++j) {
                    const int ch = (j * 32 + lane) * VW;
                    if (ch < D) load_g<VW>(grow + ch, g[j]);
                    else {
#pragma unroll
                        for (int v = 0; v < VW; ++v) g[j][v] = 0.0f;
                    }
                }
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    if (w[r] != 0.0f) {
#pragma unroll
                        for (int j = 0; j < NV; ++j)
#pragma unroll
                            for (int v = 0; v < VW; ++v) acc[r][j][v] = __fmaf_rn(w[r], g[j][v], acc[r][j][v]);
                    }
                }
            }
            // ---- 4. one vector reduction per (row, channel vector) ----
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                const int slot = c0 + warp * 8 + r;
                if (slot < U) {
                    float* drow = p.dL_dfeat + (int64_t)uid[slot] * D;
#pragma unroll
                    for (int j = 0; j < NV; ++j) {
                        const int ch = (j * 32 + lane) * VW;
                        if (ch < D) red_add<VW>(drow + ch, acc[r][j]);
                    }
                }
            }
        }
        __syncthreads();
    }
}

// plain statement: one warp per pixel
template <int NV, int VW>
__global__ void __launch_bounds__(256) backward_pixel_kernel(const BackwardParams p)
{
    const int lane = threadIdx.x & 31;
    const int64_t pix = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (pix >= (int64_t)p.cam.width * p.cam.height) return;
    const int ns = p.n_sel[pix];
    if (ns == 0) return;
    const int D = p.D, K = p.K;
    float g[NV][VW];
#pragma unroll
    for (int j = 0; j < NV; ++j) {
        const int ch = (j * 32 + lane) * VW;
        if (ch < D) load_g<VW>(p.dL_dmap + pix * D + ch, g[j]);
    }
    for (int s = 0; s < ns; ++s) {
        const int32_t id = p.sel_idx[pix * K + s];
        const float w = p.sel_w[pix * K + s];
        float* drow = p.dL_dfeat + (int64_t)id * D;
#pragma unroll
        for (int j = 0; j < NV; ++j) {
            const int ch = (j * 32 + lane) * VW;
            if (ch < D) {
                float a[VW];
#pragma unroll
                for (int v = 0; v < VW; ++v) a[v] = __fmul_rn(w, g[j][v]);
                red_add<VW>(drow + ch, a);
            }
        }
    }
}

// backward_small_kernel -- D <= 8 with D % 4 != 0 (the RGB payload, D = 3): CTA = one 16x16 tile, thread = pixel.  With so
// few channels the band kernel's lane = channel layout leaves the warp idle; here every thread walks its own selection record
// and adds w g[c] into a shared-memory hash table keyed by the Gaussian id (the tile's union is a few hundred rows), which is
// flushed with one red.global.add per (cell, channel).  An id that finds no free cell within kSmallProbe steps goes straight
// to global memory.
constexpr int kSmallCells = 2048;
constexpr int kSmallProbe = 16;
__global__ void __launch_bounds__(256) backward_small_kernel(const BackwardParams p)
{
    __shared__ int32_t s_key[kSmallCells];
    extern __shared__ __align__(16) unsigned char small_raw[];
    float* s_val = reinterpret_cast<float*>(small_raw);                  // [kSmallCells][D]
    const int tid = threadIdx.x, D = p.D, K = p.K;
    const int tile_x = blockIdx.x % p.cam.tiles_x, tile_y = blockIdx.x / p.cam.tiles_x;
    const int x = tile_x * kTile + (tid & 15), y = tile_y * kTile + (tid >> 4);
    for (int i = tid; i < kSmallCells; i += 256) s_key[i] = -1;
    for (int i = tid; i < kSmallCells * D; i += 256) s_val[i] = 0.0f;
    __syncthreads();
    if (x < p.cam.width && y < p.cam.height) {
        const int64_t pix = (int64_t)y * p.cam.width + x;
        const int ns = min(max(__ldg(p.n_sel + pix), 0), K);
        float g[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) g[c] = c < D ? __ldg(p.dL_dmap + pix * D + c) : 0.0f;
        for (int s = 0; s < ns; ++s) {
            const int32_t id = __ldg(p.sel_idx + pix * K + s);
            const float w = __ldg(p.sel_w + pix * K + s);
            if ((uint32_t)id >= (uint32_t)p.N) continue;                 // never add outside the table
            uint32_t h = hash32((uint32_t)id) & (kSmallCells - 1);
            int cell = -1;
            for (int t = 0; t < kSmallProbe; ++t) {
                const int32_t old = atomicCAS(&s_key[h], -1, id);
                if (old == -1 || old == id) { cell = (int)h; break; }
                h = (h + 1) & (kSmallCells - 1);
            }
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                if (c < D) {
                    const float a = __fmul_rn(w, g[c]);
                    if (cell >= 0) atomicAdd(&s_val[cell * D + c], a);
                    else atomicAdd(p.dL_dfeat + (int64_t)id * D + c, a);
                }
            }
        }
    }
    __syncthreads();
    for (int i = tid; i < kSmallCells * D; i += 256) {
        const int cell = i / D;
        const int32_t id = s_key[cell];
        if (id >= 0) {
            const float v = s_val[i];
            if (v != 0.0f) asm volatile("red.global.add.f32 [%0], %1;" ::"l"(p.dL_dfeat + (int64_t)id * D + (i - cell * D)), "f"(v) : "memory");
        }
    }
}

static int launch_backward_small(const BackwardParams& p, cudaStream_t st)
{
    const int T = p.cam.tiles_x * p.cam.tiles_y;
    QR_CUDA_OK(cudaFuncSetAttribute(backward_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmallCells * 8 * 4));
    backward_small_kernel<<<(unsigned)T, 256, (size_t)kSmallCells * p.D * 4, st>>>(p);
    QR_LAUNCH_OK("backward_small_kernel");
    return QR_OK;
}

static int next_pow2(int v) { int p = 1; while (p < v) p <<= 1; return p; }

template <int NV, int VW>
static int launch_backward(const BackwardParams& p, cudaStream_t st)
{
    const int T = p.cam.tiles_x * p.cam.tiles_y;
    if (p.K <= kBwdMaxK) {
        const int hs = next_pow2(2 * kBwdPx * p.K);
        const size_t smem = (size_t)kBwdPx * kBwdRows * 4 + 2 * (size_t)kBwdPx * p.K * 4 + kBwdPx * 4 +
                            2 * (size_t)hs * 4 + (size_t)kBwdPx * p.K * 4;
        auto kern = backward_band_kernel<NV, VW>;
        QR_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        kern<<<(unsigned)T * 4u, kBwdThreads, smem, st>>>(p, hs);
        QR_LAUNCH_OK("backward_band_kernel");
    } else {
        const int64_t npix = (int64_t)p.cam.width * p.cam.height;
        backward_pixel_kernel<NV, VW><<<(unsigned)((npix + 7) / 8), 256, 0, st>>>(p);
        QR_LAUNCH_OK("backward_pixel_kernel");
    }
    return QR_OK;
}

// ------------------------------------------------------------------------------------------------------------------
// qr_backward_clear: zero exactly the rows of dL_dfeat a qr_backward over the same selection adds into, so that a
// training loop re-zeroes ~|S| D floats per step instead of memset-ing the whole [N, D] table (1.02 GB at config 3,
// of which 24 MB are ever non-zero).  One CTA strides over half tiles.  Where the tcgen05 path left its numbered
// union in the workspace the rows are zeroed once per half tile; elsewhere (other D, over-full half tiles) once per
// selection record.
// ------------------------------------------------------------------------------------------------------------------
constexpr int kClearThreads = 256;
constexpr int kClearSeenCells = 1 << 20;     // de-duplication cache when qr_backward itself needs no workspace (4 MB)

__device__ __forceinline__ void clear_row(float* row, int D, int lane)
{
    if ((D & 3) == 0) {
        float4* r4 = reinterpret_cast<float4*>(row);
        for (int i = lane; i < (D >> 2); i += 32) r4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    } else {
        for (int i = lane; i < D; i += 32) row[i] = 0.0f;
    }
}


// seen[]: a direct-mapped cache of ids whose row some warp has already taken: a Gaussian is in the unions of ~10 half
// tiles, and without it every row was zeroed ~10 times (225 MB of stores for 24 MB of rows).  A collision only costs
// a repeated zeroing, never a missed one (the warp that finds another id in the cell zeroes its row).
__global__ void __launch_bounds__(kClearThreads) backward_clear_kernel(const BackwardParams p, const bool have_lists,
                                                                       int32_t* __restrict__ seen, const int seen_mask)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int num_half = p.cam.tiles_x * p.cam.tiles_y * 2;
    // a workspace that does not hold the lists of this camera and K (fresh memory, another frame size) is not trusted:
    // fall back to the selection records, which are this call's own arguments
    const bool lists = have_lists && sel_stamp_ok(p.sl.stamp, p.cam, p.K);
    for (int ht = blockIdx.x; ht < num_half; ht += gridDim.x) {
        const int tile = ht >> 1;
        const int x0 = (tile % p.cam.tiles_x) * kTile, y0 = (tile / p.cam.tiles_x) * kTile + (ht & 1) * 8;
        if (y0 >= p.cam.height) continue;
        int U = 0, flagged = 1;
        if (lists) {
            const int32_t* hd = p.sl.hdr + (size_t)ht * kHdrWords;
            U = hd[4]; flagged = hd[5];
            if (flagged == 0 && U == 0) continue;                 // nothing selected in this half tile
        }
        if (flagged == 0) {                                       // numbered union: one pass over its rows
            const int32_t* uid = p.sl.uid + (size_t)ht * p.sl.ucap;
            for (int r0 = 0; r0 < U; r0 += kClearThreads) {         // thread = union row: claim it, then the warp zeroes the claimed rows
                const int r = r0 + (int)threadIdx.x;
                int32_t id = -1;
                if (r < U) {
                    id = uid[r];
                    if ((uint32_t)id >= (uint32_t)p.N) id = -1;    // never write outside the table
                    else if (seen && atomicExch(&seen[hash32((uint32_t)id) & seen_mask], id) == id) id = -1;   // already taken
                }
                uint32_t todo = __ballot_sync(0xffffffffu, id >= 0);
                while (todo) {
                    const int src = __ffs(todo) - 1;
                    todo &= todo - 1;
                    clear_row(p.dL_dfeat + (int64_t)__shfl_sync(0xffffffffu, id, src) * p.D, p.D, lane);
                }
            }
        } else {                                                  // every record of the 16 x 8 pixels
            for (int q = warp; q < 128; q += kClearThreads / 32) {      // warp = pixel, lane = record
                const int x = x0 + (q & 15), y = y0 + (q >> 4);
                if (x >= p.cam.width || y >= p.cam.height) continue;
                const int64_t pix = (int64_t)y * p.cam.width + x;
                const int ns = max(0, min(p.K, __ldg(p.n_sel + pix)));
                for (int s0 = 0; s0 < ns; s0 += 32) {
                    int32_t id = -1;
                    if (s0 + lane < ns) {
                        id = __ldg(p.sel_idx + pix * p.K + s0 + lane);
                        if ((uint32_t)id >= (uint32_t)p.N) id = -1;    // never write outside the table
                        else if (seen && atomicExch(&seen[hash32((uint32_t)id) & seen_mask], id) == id) id = -1;   // already taken
                    }
                    uint32_t todo = __ballot_sync(0xffffffffu, id >= 0);
                    while (todo) {
                        const int src = __ffs(todo) - 1;
                        todo &= todo - 1;
                        clear_row(p.dL_dfeat + (int64_t)__shfl_sync(0xffffffffu, id, src) * p.D, p.D, lane);
                    }
                }
            }
        }
    }
}

}  // namespace qr

extern "C" int qr_backward_clear(const qr_camera* cam, int32_t K, int32_t D, int64_t N, const int32_t* sel_idx,
                                 const int32_t* n_sel, float* dL_dfeat, void* ws, size_t ws_bytes, void* stream)
{
    using namespace qr;
    if (int rc = check_cam(cam)) return rc;
    if (K < 1) return fail(QR_ERR_INVALID_ARG, "qr_backward_clear: K = %d < 1", K);
    if (K > QR_MAX_K) return fail(QR_ERR_UNSUPPORTED, "qr_backward_clear: K = %d > QR_MAX_K", K);
    if (D < 1) return fail(QR_ERR_INVALID_ARG, "qr_backward_clear: D = %d < 1", D);
    if (D > QR_MAX_D) return fail(QR_ERR_UNSUPPORTED, "qr_backward_clear: D = %d > QR_MAX_D", D);
    if (N < 0) return fail(QR_ERR_INVALID_ARG, "qr_backward_clear: N < 0");
    if (!sel_idx || !n_sel) return fail(QR_ERR_NULL_POINTER, "qr_backward_clear: NULL input");
    if (N == 0) return QR_OK;
    if (!dL_dfeat) return fail(QR_ERR_NULL_POINTER, "qr_backward_clear: dL_dfeat is NULL");
    if (!aligned16(dL_dfeat)) return fail(QR_ERR_MISALIGNED, "qr_backward_clear: 16-byte alignment");
    BackwardParams p;
    p.cam = make_cam(cam); p.K = K; p.D = D; p.N = N;
    p.sel_idx = sel_idx; p.sel_w = nullptr; p.n_sel = n_sel; p.dL_dmap = nullptr; p.dL_dfeat = dL_dfeat;
    int seen_cells = 0;
    int32_t* seen = nullptr;
    bool have_lists = false;
    if (!ws) return fail(QR_ERR_NULL_POINTER, "qr_backward_clear: workspace is NULL");
    if (backward_mma_supported(K, D)) {
        if (int rc = backward_mma_workspace_view(p, ws, ws_bytes, &seen, &seen_cells)) return rc;
        have_lists = true;
    } else {                                    // no numbered unions: the workspace is only the de-duplication cache
        if (ws_bytes < (size_t)kClearSeenCells * 4) return fail(QR_ERR_WORKSPACE_TOO_SMALL, "qr_backward_clear: workspace %zu < %zu bytes", ws_bytes, (size_t)kClearSeenCells * 4);
        if (!aligned16(ws)) return fail(QR_ERR_MISALIGNED, "qr_backward_clear: workspace alignment");
        seen = static_cast<int32_t*>(ws);
        seen_cells = kClearSeenCells;
    }
    QR_CUDA_OK(cudaMemsetAsync(seen, 0xFF, (size_t)seen_cells * 4, (cudaStream_t)stream));
    const int sms = sm_count();
    const int num_half = p.cam.tiles_x * p.cam.tiles_y * 2;
    backward_clear_kernel<<<(unsigned)min(num_half, sms * 8), kClearThreads, 0, (cudaStream_t)stream>>>(p, have_lists, seen, seen_cells - 1);
    QR_LAUNCH_OK("backward_clear_kernel");
    return QR_OK;
}

extern "C" size_t qr_backward_workspace_bytes(const qr_camera* cam, int32_t K, int32_t D)
{
    if (!cam || cam->width < 1 || cam->height < 1) return 0;
    return qr::backward_mma_supported(K, D) ? qr::backward_mma_workspace_bytes(qr::make_cam(cam), K)
                                            : (size_t)qr::kClearSeenCells * 4;      // used by qr_backward_clear only
}

extern "C" int qr_backward(const qr_camera* cam, int32_t K, int32_t D, int64_t N, const int32_t* sel_idx,
                           const float* sel_w, const int32_t* n_sel, const float* dL_dmap, float* dL_dfeat, void* ws,
                           size_t ws_bytes, void* stream)
{
    using namespace qr;
    if (int rc = check_cam(cam)) return rc;
    if (K < 1) return fail(QR_ERR_INVALID_ARG, "qr_backward: K = %d < 1", K);
    if (K > QR_MAX_K) return fail(QR_ERR_UNSUPPORTED, "qr_backward: K = %d > QR_MAX_K", K);
    if (D < 1) return fail(QR_ERR_INVALID_ARG, "qr_backward: D = %d < 1", D);
    if (D > QR_MAX_D) return fail(QR_ERR_UNSUPPORTED, "qr_backward: D = %d > QR_MAX_D", D);
    if (D % 4 != 0 && D > 128) return fail(QR_ERR_UNSUPPORTED, "qr_backward: D %% 4 != 0 is only supported for D <= 128");
    if (N < 0) return fail(QR_ERR_INVALID_ARG, "qr_backward: N < 0");
    if (!sel_idx || !sel_w || !n_sel || !dL_dmap) return fail(QR_ERR_NULL_POINTER, "qr_backward: NULL input");
    if (N == 0) return QR_OK;
    if (!dL_dfeat) return fail(QR_ERR_NULL_POINTER, "qr_backward: dL_dfeat is NULL");
    if (!aligned16(dL_dmap) || !aligned16(dL_dfeat)) return fail(QR_ERR_MISALIGNED, "qr_backward: 16-byte alignment");
    BackwardParams p;
    p.cam = make_cam(cam); p.K = K; p.D = D; p.N = N;
    p.sel_idx = sel_idx; p.sel_w = sel_w; p.n_sel = n_sel; p.dL_dmap = dL_dmap; p.dL_dfeat = dL_dfeat;
    cudaStream_t st = (cudaStream_t)stream;
    if (backward_mma_supported(K, D)) return launch_backward_mma(p, ws, ws_bytes, st, false);
    if (backward_tile_supported(K, D)) return launch_backward_tile(p, st);
    // D % 4 == 0 never reaches this point (backward_tile_supported takes it): what is left is D % 4 != 0, D <= 128
    if (D <= 8) return launch_backward_small(p, st);
    switch ((D + 31) / 32) {
        case 1: return launch_backward<1, 1>(p, st);
        case 2: return launch_backward<2, 1>(p, st);
        case 3: return launch_backward<3, 1>(p, st);
        default: return launch_backward<4, 1>(p, st);
    }
}

extern "C" int qr_backward_lists(const qr_camera* cam, int32_t K, int32_t D, int64_t N, void* fwd_ws, size_t fwd_ws_bytes,
                                 const float* dL_dmap, float* dL_dfeat, void* stream)
{
    using namespace qr;
    if (int rc = check_cam(cam)) return rc;
    if (K < 1) return fail(QR_ERR_INVALID_ARG, "qr_backward_lists: K = %d < 1", K);
    if (K > QR_MAX_K) return fail(QR_ERR_UNSUPPORTED, "qr_backward_lists: K = %d > QR_MAX_K", K);
    if (!backward_mma_supported(K, D))
        return fail(QR_ERR_UNSUPPORTED, "qr_backward_lists: needs D %% 32 == 0 (or D < 32 with D %% 4 == 0), D <= 512 (D = %d): use qr_backward", D);
    if (N < 0) return fail(QR_ERR_INVALID_ARG, "qr_backward_lists: N < 0");
    if (!fwd_ws || !dL_dmap) return fail(QR_ERR_NULL_POINTER, "qr_backward_lists: NULL input");
    if (N == 0) return QR_OK;
    if (!dL_dfeat) return fail(QR_ERR_NULL_POINTER, "qr_backward_lists: dL_dfeat is NULL");
    if (!aligned16(dL_dmap) || !aligned16(dL_dfeat)) return fail(QR_ERR_MISALIGNED, "qr_backward_lists: 16-byte alignment");
    BackwardParams p;
    p.cam = make_cam(cam); p.K = K; p.D = D; p.N = N;
    p.sel_idx = nullptr; p.sel_w = nullptr; p.n_sel = nullptr; p.dL_dmap = dL_dmap; p.dL_dfeat = dL_dfeat;
    return launch_backward_mma(p, fwd_ws, fwd_ws_bytes, (cudaStream_t)stream, true);
}

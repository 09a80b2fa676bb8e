// qr_bin.cu -- tiling stage: prefix sum of tiles touched, tile-intersection duplication, stable LSD radix sort of
// (tile, depth) keys, per-tile ranges.  PAPER.md:80 "(1) tiling strategy", :86 "ordered sequence of indices";
// SPEC.md:139-147, :167-168; reading R6 (ascending depth, ties by ascending Gaussian index).
//
// Everything is integer work: depth > znear > 0, so the IEEE bit pattern of depth orders like the float.
// All kernels are hand-written (no CUB): scan = reduce / scan-of-sums / scan-and-add; sort = per pass
// {block digit histograms, exclusive scan of the digit-major histogram table, stable scatter}.
#include "qr_common.cuh"

namespace qr {

// ------------------------------------------------------------------------------------------------------------
// inclusive scan of uint32 -> uint64, 2048 elements per block
// ------------------------------------------------------------------------------------------------------------
constexpr int kScanThreads = 256;
constexpr int kScanItems = 8;
constexpr int kScanChunk = kScanThreads * kScanItems;

__device__ __forceinline__ uint64_t block_exclusive_scan_u64(uint64_t v, uint64_t* total, uint64_t* warp_sums)
{
    // returns the exclusive prefix of v over the block (256 threads); *total = block sum (valid in all threads)
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint64_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint64_t n = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += n;
    }
    if (lane == 31) warp_sums[warp] = inc;
    __syncthreads();
    uint64_t base = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < kScanThreads / 32; ++w) {
        const uint64_t s = warp_sums[w];
        if (w < warp) base += s;
        tot += s;
    }
    __syncthreads();
    *total = tot;
    return base + inc - v;
}

__global__ void __launch_bounds__(kScanThreads)
scan_reduce_kernel(const uint32_t* __restrict__ in, int64_t N, uint64_t* __restrict__ block_sums)
{
    __shared__ uint64_t warp_sums[kScanThreads / 32];
    const int64_t base = (int64_t)blockIdx.x * kScanChunk;
    uint64_t s = 0;
#pragma unroll
    for (int j = 0; j < kScanItems; ++j) {
        const int64_t i = base + (int64_t)j * kScanThreads + threadIdx.x;
        if (i < N) s += in[i];
    }
    uint64_t tot;
    block_exclusive_scan_u64(s, &tot, warp_sums);
    if (threadIdx.x == 0) block_sums[blockIdx.x] = tot;
}

// one block: exclusive scan of block_sums[nb] in place
__global__ void __launch_bounds__(kScanThreads)
scan_sums_kernel(uint64_t* __restrict__ block_sums, int64_t nb)
{
    __shared__ uint64_t warp_sums[kScanThreads / 32];
    uint64_t carry = 0;
    for (int64_t b0 = 0; b0 < nb; b0 += kScanThreads) {
        const int64_t i = b0 + threadIdx.x;
        const uint64_t v = i < nb ? block_sums[i] : 0;
        uint64_t tot;
        const uint64_t ex = block_exclusive_scan_u64(v, &tot, warp_sums);
        if (i < nb) block_sums[i] = carry + ex;
        carry += tot;
    }
}

__global__ void __launch_bounds__(kScanThreads)
scan_apply_kernel(const uint32_t* __restrict__ in, int64_t N, const uint64_t* __restrict__ block_sums,
                  uint64_t* __restrict__ out)
{
    __shared__ uint64_t warp_sums[kScanThreads / 32];
    // thread t owns the kScanItems consecutive elements base + t*kScanItems .. (order-preserving layout)
    const int64_t base = (int64_t)blockIdx.x * kScanChunk + (int64_t)threadIdx.x * kScanItems;
    uint32_t v[kScanItems];
    uint64_t s = 0;
#pragma unroll
    for (int j = 0; j < kScanItems; ++j) {
        v[j] = (base + j < N) ? in[base + j] : 0u;
        s += v[j];
    }
    uint64_t tot;
    uint64_t run = block_sums[blockIdx.x] + block_exclusive_scan_u64(s, &tot, warp_sums);
#pragma unroll
    for (int j = 0; j < kScanItems; ++j) {
        run += v[j];
        if (base + j < N) out[base + j] = run;
    }
}

// ------------------------------------------------------------------------------------------------------------
// duplication: one key per (Gaussian, tile of its rectangle); value = Gaussian id.  Emitted in Gaussian-id order
// (offsets is a scan in id order), so a stable sort breaks depth ties by ascending id (R6).
// One warp per 32 Gaussians; lanes stride over each rectangle's tiles so a screen-filling footprint does not
// serialise on one thread.
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
duplicate_kernel(int64_t N, int32_t tiles_x, const float* __restrict__ depth, const int4* __restrict__ tile_rect,
                 const uint64_t* __restrict__ offsets, uint64_t* __restrict__ keys, uint32_t* __restrict__ vals)
{
    const int lane = threadIdx.x & 31;
    const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x - lane);   // first Gaussian of this warp
    int4 r = make_int4(0, 0, 0, 0);
    uint64_t end = 0;
    uint32_t dbits = 0;
    const int64_t i = warp0 + lane;
    if (i < N) {
        r = tile_rect[i];
        end = offsets[i];
        dbits = __float_as_uint(depth[i]);
    }
    const int w = r.z - r.x, h = r.w - r.y;
    const uint32_t cnt = (uint32_t)(w * h);
    for (int src = 0; src < 32; ++src) {
        const uint32_t c = __shfl_sync(0xffffffffu, cnt, src);
        if (c == 0) continue;
        const int x0 = __shfl_sync(0xffffffffu, r.x, src), y0 = __shfl_sync(0xffffffffu, r.y, src);
        const int ww = __shfl_sync(0xffffffffu, w, src);
        const uint64_t e = __shfl_sync(0xffffffffu, end, src);
        const uint32_t db = __shfl_sync(0xffffffffu, dbits, src);
        const uint64_t start = e - c;
        for (uint32_t j = lane; j < c; j += 32) {
            const int ty = y0 + (int)(j / (uint32_t)ww), tx = x0 + (int)(j % (uint32_t)ww);
            const uint64_t tile = (uint64_t)(ty * tiles_x + tx);
            keys[start + j] = (tile << 32) | db;
            vals[start + j] = (uint32_t)(warp0 + src);
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// LSD radix sort, 8-bit digits.  Block = 256 threads = 8 warps; a block owns kSortChunk consecutive keys, warp w
// owns the 512 consecutive keys [w*512, w*512+512) of it, lane l holds keys r*32 + l, r = 0..15 (coalesced).
// ------------------------------------------------------------------------------------------------------------
constexpr int kSortThreads = 256;
constexpr int kSortRounds = 16;
constexpr int kSortWarpKeys = 32 * kSortRounds;           // 512
constexpr int kSortChunk = (kSortThreads / 32) * kSortWarpKeys;   // 4096

__global__ void __launch_bounds__(kSortThreads)
sort_hist_kernel(const uint64_t* __restrict__ keys, int64_t M, int shift, uint32_t* __restrict__ hist, int nblocks)
{
    __shared__ uint32_t h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * kSortChunk;
#pragma unroll 4
    for (int j = 0; j < kSortChunk / kSortThreads; ++j) {
        const int64_t i = base + (int64_t)j * kSortThreads + threadIdx.x;
        if (i < M) atomicAdd(&h[(uint32_t)(keys[i] >> shift) & 255u], 1u);
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * nblocks + blockIdx.x] = h[threadIdx.x];   // digit-major table
}

// one block of 1024 threads: exclusive scan of the digit-major table hist[256 * nblocks] in place
__global__ void __launch_bounds__(1024)
sort_scan_kernel(uint32_t* __restrict__ hist, int64_t n)
{
    __shared__ uint32_t warp_sums[32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t carry = 0;
    for (int64_t b0 = 0; b0 < n; b0 += 1024 * 4) {
        const int64_t i0 = b0 + (int64_t)threadIdx.x * 4;
        uint32_t v[4], s = 0;
#pragma unroll
        for (int j = 0; j < 4; ++j) { v[j] = (i0 + j < n) ? hist[i0 + j] : 0u; s += v[j]; }
        uint32_t inc = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) warp_sums[warp] = inc;
        __syncthreads();
        uint32_t wbase = 0, tot = 0;
        for (int w = 0; w < 32; ++w) { const uint32_t x = warp_sums[w]; if (w < warp) wbase += x; tot += x; }
        __syncthreads();
        uint32_t run = carry + wbase + inc - s;
#pragma unroll
        for (int j = 0; j < 4; ++j) { if (i0 + j < n) hist[i0 + j] = run; run += v[j]; }
        carry += tot;
    }
}

__global__ void __launch_bounds__(kSortThreads)
sort_scatter_kernel(const uint64_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in, int64_t M, int shift,
                    const uint32_t* __restrict__ hist_scanned, int nblocks, uint64_t* __restrict__ keys_out,
                    uint32_t* __restrict__ vals_out)
{
    __shared__ uint32_t wofs[kSortThreads / 32][256];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int j = threadIdx.x; j < (kSortThreads / 32) * 256; j += kSortThreads) (&wofs[0][0])[j] = 0;
    __syncthreads();

    const int64_t wbase = (int64_t)blockIdx.x * kSortChunk + (int64_t)warp * kSortWarpKeys;
    uint64_t k[kSortRounds];
    uint32_t v[kSortRounds];
#pragma unroll
    for (int r = 0; r < kSortRounds; ++r) {
        const int64_t i = wbase + r * 32 + lane;
        if (i < M) { k[r] = keys_in[i]; v[r] = vals_in[i]; } else { k[r] = 0; v[r] = 0; }
    }
    // warp-private digit histogram
#pragma unroll
    for (int r = 0; r < kSortRounds; ++r)
        if (wbase + r * 32 + lane < M) atomicAdd(&wofs[warp][(uint32_t)(k[r] >> shift) & 255u], 1u);
    __syncthreads();
    {   // digit d = threadIdx.x: exclusive prefix over warps + this block's global base
        const int d = threadIdx.x;
        uint32_t run = hist_scanned[(size_t)d * nblocks + blockIdx.x];
#pragma unroll
        for (int w = 0; w < kSortThreads / 32; ++w) { const uint32_t c = wofs[w][d]; wofs[w][d] = run; run += c; }
    }
    __syncthreads();
    // stable placement: rounds in order, lanes in order within a round
#pragma unroll
    for (int r = 0; r < kSortRounds; ++r) {
        const bool valid = wbase + r * 32 + lane < M;
        const uint32_t d = valid ? ((uint32_t)(k[r] >> shift) & 255u) : 256u + lane;   // invalid lanes match nobody
        const uint32_t peers = __match_any_sync(0xffffffffu, d);
        const uint32_t rank = __popc(peers & ((1u << lane) - 1u));
        uint32_t pos = 0;
        if (valid) pos = wofs[warp][d] + rank;
        __syncwarp();
        if (valid && rank == 0) wofs[warp][d] += __popc(peers);
        __syncwarp();
        if (valid) { keys_out[pos] = k[r]; vals_out[pos] = v[r]; }
    }
}

// per-tile ranges by binary search of the sorted keys: start(t) = #keys with tile id < t
__global__ void __launch_bounds__(256)
tile_range_kernel(const uint64_t* __restrict__ keys, int64_t M, int32_t T, int32_t* __restrict__ tile_range)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t > T) return;
    const uint64_t target = (uint64_t)t << 32;
    int64_t lo = 0, hi = M;
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if (keys[mid] < target) lo = mid + 1; else hi = mid;
    }
    if (t < T) tile_range[2 * t] = (int32_t)lo;
    if (t > 0) tile_range[2 * (t - 1) + 1] = (int32_t)lo;
}

struct BinLayout {
    size_t keys0, keys1, vals1, hist, sums, total;
    int nblocks_sort;
    int64_t nblocks_scan;
};

static BinLayout bin_layout(int64_t N, int64_t M, int32_t /*T*/)
{
    BinLayout L;
    const size_t m = (size_t)(M > 0 ? M : 1);
    L.nblocks_sort = (int)((m + kSortChunk - 1) / kSortChunk);
    L.nblocks_scan = (N + kScanChunk - 1) / kScanChunk;
    if (L.nblocks_scan < 1) L.nblocks_scan = 1;
    size_t o = 0;
    L.keys0 = o; o = align_up(o + m * 8, 256);
    L.keys1 = o; o = align_up(o + m * 8, 256);
    L.vals1 = o; o = align_up(o + m * 4, 256);
    L.hist = o;  o = align_up(o + (size_t)256 * L.nblocks_sort * 4, 256);
    L.sums = o;  o = align_up(o + (size_t)L.nblocks_scan * 8, 256);
    L.total = o;
    return L;
}

}  // namespace qr

extern "C" size_t qr_bin_workspace_bytes(int64_t N, int64_t M_capacity, int32_t num_tiles)
{
    if (N < 0 || M_capacity < 0) return 0;
    return qr::bin_layout(N, M_capacity, num_tiles).total;
}

extern "C" int qr_bin_count(int64_t N, const uint32_t* tiles_touched, uint64_t* offsets, int64_t* M_host,
                            void* ws, size_t ws_bytes, void* stream)
{
    using namespace qr;
    if (N < 0) return fail(QR_ERR_INVALID_ARG, "N = %lld < 0", (long long)N);
    if (!M_host) return fail(QR_ERR_NULL_POINTER, "qr_bin_count: M_host is NULL");
    if (N == 0) { *M_host = 0; return QR_OK; }
    if (!tiles_touched || !offsets || !ws) return fail(QR_ERR_NULL_POINTER, "qr_bin_count: NULL array");
    const BinLayout L = bin_layout(N, 0, 0);
    if (ws_bytes < L.sums + (size_t)L.nblocks_scan * 8)
        return fail(QR_ERR_WORKSPACE_TOO_SMALL, "qr_bin_count: workspace %zu < %zu bytes", ws_bytes,
                    L.sums + (size_t)L.nblocks_scan * 8);
    cudaStream_t st = (cudaStream_t)stream;
    uint64_t* sums = reinterpret_cast<uint64_t*>(static_cast<char*>(ws) + L.sums);
    const unsigned nb = (unsigned)L.nblocks_scan;
    scan_reduce_kernel<<<nb, kScanThreads, 0, st>>>(tiles_touched, N, sums);
    QR_LAUNCH_OK("scan_reduce_kernel");
    scan_sums_kernel<<<1, kScanThreads, 0, st>>>(sums, L.nblocks_scan);
    QR_LAUNCH_OK("scan_sums_kernel");
    scan_apply_kernel<<<nb, kScanThreads, 0, st>>>(tiles_touched, N, sums, offsets);
    QR_LAUNCH_OK("scan_apply_kernel");
    uint64_t m = 0;
    QR_CUDA_OK(cudaMemcpyAsync(&m, offsets + (N - 1), sizeof(uint64_t), cudaMemcpyDeviceToHost, st));
    QR_CUDA_OK(cudaStreamSynchronize(st));
    *M_host = (int64_t)m;
    return QR_OK;
}

extern "C" int qr_bin_sort(const qr_camera* cam, int64_t N, int64_t M, const float* depth, const int32_t* tile_rect,
                           const uint64_t* offsets, uint32_t* isect_gauss, int32_t* tile_range, void* ws,
                           size_t ws_bytes, void* stream)
{
    using namespace qr;
    if (int rc = check_cam(cam)) return rc;
    if (N < 0 || M < 0) return fail(QR_ERR_INVALID_ARG, "N or M < 0");
    if (M >= (int64_t(1) << 31)) return fail(QR_ERR_CAPACITY, "M = %lld >= 2^31 intersections", (long long)M);
    if (!tile_range) return fail(QR_ERR_NULL_POINTER, "qr_bin_sort: tile_range is NULL");
    const Cam k = make_cam(cam);
    const int32_t T = k.tiles_x * k.tiles_y;
    cudaStream_t st = (cudaStream_t)stream;
    if (M == 0 || N == 0) {
        QR_CUDA_OK(cudaMemsetAsync(tile_range, 0, sizeof(int32_t) * 2 * (size_t)T, st));
        return QR_OK;
    }
    if (!depth || !tile_rect || !offsets || !isect_gauss || !ws)
        return fail(QR_ERR_NULL_POINTER, "qr_bin_sort: NULL array");
    if (!aligned16(tile_rect) || !aligned16(ws)) return fail(QR_ERR_MISALIGNED, "qr_bin_sort: tile_rect / ws alignment");
    const BinLayout L = bin_layout(N, M, T);
    if (ws_bytes < L.total)
        return fail(QR_ERR_WORKSPACE_TOO_SMALL, "qr_bin_sort: workspace %zu < %zu bytes", ws_bytes, L.total);
    char* w = static_cast<char*>(ws);
    uint64_t* keys[2] = { reinterpret_cast<uint64_t*>(w + L.keys0), reinterpret_cast<uint64_t*>(w + L.keys1) };
    uint32_t* vals[2] = { isect_gauss, reinterpret_cast<uint32_t*>(w + L.vals1) };
    uint32_t* hist = reinterpret_cast<uint32_t*>(w + L.hist);

    int tile_bits = 0;
    while ((int64_t(1) << tile_bits) < T) ++tile_bits;
    const int passes = (32 + tile_bits + 7) / 8;
    int cur = (passes % 2 == 0) ? 0 : 1;   // so that the last pass writes vals[0] = isect_gauss

    duplicate_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(N, k.tiles_x, depth,
                                                                 reinterpret_cast<const int4*>(tile_rect), offsets,
                                                                 keys[cur], vals[cur]);
    QR_LAUNCH_OK("duplicate_kernel");
    const int nb = L.nblocks_sort;
    for (int p = 0; p < passes; ++p) {
        const int shift = 8 * p;
        sort_hist_kernel<<<nb, kSortThreads, 0, st>>>(keys[cur], M, shift, hist, nb);
        QR_LAUNCH_OK("sort_hist_kernel");
        sort_scan_kernel<<<1, 1024, 0, st>>>(hist, (int64_t)256 * nb);
        QR_LAUNCH_OK("sort_scan_kernel");
        sort_scatter_kernel<<<nb, kSortThreads, 0, st>>>(keys[cur], vals[cur], M, shift, hist, nb, keys[cur ^ 1],
                                                         vals[cur ^ 1]);
        QR_LAUNCH_OK("sort_scatter_kernel");
        cur ^= 1;
    }
    // cur == 0 here: sorted ids are in isect_gauss, sorted keys in keys[0]
    tile_range_kernel<<<(unsigned)((T + 1 + 255) / 256), 256, 0, st>>>(keys[cur], M, T, tile_range);
    QR_LAUNCH_OK("tile_range_kernel");
    return QR_OK;
}

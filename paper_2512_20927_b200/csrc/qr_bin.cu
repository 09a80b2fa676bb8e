// qr_bin.cu -- tiling stage: prefix sum of tiles touched, tile-intersection duplication, sort by (tile, depth, id),
// per-tile ranges.  PAPER.md:80 "(1) tiling strategy", :86 "ordered sequence of indices"; SPEC.md:139-147, :167-168;
// reading R6 (ascending depth, ties by ascending Gaussian index).
//
// Everything is integer work: depth > znear > 0, so the IEEE bit pattern of depth orders like the float.
// All kernels are hand-written (no CUB): scan = reduce / scan-of-sums / scan-and-add; sort = most-significant-digit
// radix pass over the tile field (count, scan, scatter) + a shared-memory bitonic network per tile bucket.
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
// Sort by (tile, depth, id) = one most-significant-digit radix pass over the tile field (a counting sort with one
// bucket per tile: count, exclusive scan, scatter) followed by an in-shared-memory sort of every bucket on its
// 64-bit (depth bits << 32 | Gaussian id) keys.  Those keys are unique, so the order inside a bucket does not
// depend on the order in which the scatter filled it: ties in depth fall to the ascending id (R6) by construction,
// and the result is bit-identical from run to run.  6 launches per frame instead of the 20 of an 8-bit LSD sort
// over the whole 43-bit key (ncu launch list in profiles/: the LSD passes were launch-latency bound at M = 5e5).
// ------------------------------------------------------------------------------------------------------------

// One warp per 32 Gaussians; lanes stride over each rectangle's tiles so a screen-filling footprint does not
// serialise on one thread.  SCATTER = false: count[slot] += 1.  SCATTER = true: keys[cursor[slot]++] = key.
// A tile has kSubBuckets counters (slot = tile * kSubBuckets + Gaussian id % kSubBuckets), contiguous in the scan, so
// a crowded tile's atomics spread over kSubBuckets L2 addresses instead of serialising on one (a same-address
// atomic chain of ~1,500 was the whole cost of the first version of this kernel).
constexpr int kSubBuckets = 16;
template <bool SCATTER>
__global__ void __launch_bounds__(256)
tile_bucket_kernel(int64_t N, int32_t tiles_x, const float* __restrict__ depth, const int4* __restrict__ tile_rect,
                   uint32_t* __restrict__ counter, uint64_t* __restrict__ keys, uint32_t capacity)
{
    const int lane = threadIdx.x & 31;
    const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x - lane);   // first Gaussian of this warp
    int4 r = make_int4(0, 0, 0, 0);
    uint32_t dbits = 0;
    const int64_t i = warp0 + lane;
    if (i < N) {
        r = tile_rect[i];
        if (SCATTER) dbits = __float_as_uint(depth[i]);
    }
    const int w = r.z - r.x, h = r.w - r.y;
    const uint32_t cnt = (uint32_t)(w * h);
    uint32_t todo = __ballot_sync(0xffffffffu, cnt != 0u);
    while (todo) {
        const int src = __ffs(todo) - 1;
        todo &= todo - 1;
        const uint32_t c = __shfl_sync(0xffffffffu, cnt, src);
        const int x0 = __shfl_sync(0xffffffffu, r.x, src), y0 = __shfl_sync(0xffffffffu, r.y, src);
        const int ww = __shfl_sync(0xffffffffu, w, src);
        const uint32_t db = __shfl_sync(0xffffffffu, dbits, src);
        const uint64_t key = ((uint64_t)db << 32) | (uint64_t)(uint32_t)(warp0 + src);
        for (uint32_t j = lane; j < c; j += 32) {
            const int ty = y0 + (int)(j / (uint32_t)ww), tx = x0 + (int)(j % (uint32_t)ww);
            const int slot = (ty * tiles_x + tx) * kSubBuckets + (int)((uint32_t)(warp0 + src) % kSubBuckets);
            if (SCATTER) {
                const uint32_t pos = atomicAdd(&counter[slot], 1u);
                if (pos < capacity) keys[pos] = key;           // M was only an upper bound and it was too small: dropped
            }
            else atomicAdd(&counter[slot], 1u);
        }
    }
}

// one block of 1024 threads, thread = tile: exclusive scan of the T * kSubBuckets slot counts -> cursors in place;
// tile_range[t] = [cursor of the tile's first slot, end of its last slot)
__global__ void __launch_bounds__(1024)
tile_scan_kernel(uint32_t* __restrict__ counter, int32_t T, int32_t* __restrict__ tile_range, uint32_t capacity,
                 int64_t* __restrict__ found)
{
    static_assert(kSubBuckets % 4 == 0, "slots are read as uint4");
    __shared__ uint32_t warp_sums[32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t carry = 0;
    for (int32_t t0 = 0; t0 < T; t0 += 1024) {
        const int32_t t = t0 + (int32_t)threadIdx.x;
        uint32_t v[kSubBuckets], s = 0;
        uint4* slots = reinterpret_cast<uint4*>(counter + (size_t)t * kSubBuckets);
#pragma unroll
        for (int j = 0; j < kSubBuckets / 4; ++j) {
            const uint4 q = t < T ? slots[j] : make_uint4(0u, 0u, 0u, 0u);
            v[4 * j] = q.x; v[4 * j + 1] = q.y; v[4 * j + 2] = q.z; v[4 * j + 3] = q.w;
            s += q.x + q.y + q.z + q.w;
        }
        uint32_t inc = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += u;
        }
        if (lane == 31) warp_sums[warp] = inc;
        __syncthreads();
        const uint32_t ws = warp_sums[lane];
        uint32_t winc = ws;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += u;
        }
        const uint32_t wbase = __shfl_sync(0xffffffffu, winc - ws, warp);
        const uint32_t tot = __shfl_sync(0xffffffffu, winc, 31);
        __syncthreads();
        uint32_t run = carry + wbase + inc - s;
        if (t < T) {
            tile_range[2 * t] = (int32_t)min(run, capacity);            // lists are truncated at the caller's capacity
            tile_range[2 * t + 1] = (int32_t)min(run + s, capacity);
#pragma unroll
            for (int j = 0; j < kSubBuckets / 4; ++j) {
                uint4 q;
                q.x = run; run += v[4 * j];
                q.y = run; run += v[4 * j + 1];
                q.z = run; run += v[4 * j + 2];
                q.w = run; run += v[4 * j + 3];
                slots[j] = q;
            }
        }
        carry += tot;
    }
    if (threadIdx.x == 0) *found = (int64_t)carry;                       // intersections found (> capacity: truncated)
}

// bitonic network over n2 (a power of two, >= 32 per warp) keys in shared memory; every thread of the block takes
// part.  Warp w owns the contiguous chunk [w n2 / W, (w + 1) n2 / W): a compare-exchange step of stride j < chunk
// stays inside the chunk and needs only __syncwarp; block barriers remain for the log2(W) largest strides of a merge
// (6 of the 45 steps at n2 = 512 with 8 warps) -- the network was bound by barrier stalls before (profiles/README.md).
__device__ __forceinline__ void bitonic_sort_smem(uint64_t* s, int n2)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int chunk = min(max(n2 / nwarps, 64), n2);        // keys per warp-local chunk (a power of two)
    const int nchunks = n2 / chunk;                         // <= nwarps; warps beyond it idle in the local steps
    bool local_before = false;
    for (int k = 2; k <= n2; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            if (j >= chunk) {                               // pairs span chunks: whole block, block barrier
                if (local_before) __syncthreads();
                for (int idx = threadIdx.x; idx < (n2 >> 1); idx += blockDim.x) {
                    const int i = ((idx & ~(j - 1)) << 1) | (idx & (j - 1));
                    const int l = i | j;
                    const uint64_t a = s[i], b = s[l];
                    if ((a > b) == ((i & k) == 0)) { s[i] = b; s[l] = a; }
                }
                __syncthreads();
                local_before = false;
            } else {
                if (warp < nchunks) {
                    const int base = warp * chunk;
                    for (int idx = lane; idx < (chunk >> 1); idx += 32) {
                        const int i = base + (((idx & ~(j - 1)) << 1) | (idx & (j - 1)));
                        const int l = i | j;
                        const uint64_t a = s[i], b = s[l];
                        if ((a > b) == ((i & k) == 0)) { s[i] = b; s[l] = a; }
                    }
                }
                __syncwarp();
                local_before = true;
            }
        }
    }
    __syncthreads();
}

constexpr int kSmallBucket = 2048;          // keys sorted by tile_sort_kernel<small> (16 KB of shared memory)
constexpr int kBigBucket = 8192;            // keys per shared-memory run of tile_sort_kernel<big> (64 KB: two CTAs per SM)
constexpr uint64_t kKeyInf = ~uint64_t(0);
constexpr int kBigSmem = kBigBucket * 8 + 32 * 256 * 4;      // a run of keys + the radix sort's per-warp digit counters

// Register-blocked bitonic network for one bucket of THREADS x E keys: thread t holds keys
// t E .. t E + E - 1.  Strides below E are compare-exchanges inside a thread, strides below 32 E are exchanged with
// __shfl_xor, and only the three largest strides of the last three merges (6 steps of the 36..66) go through shared
// memory.  The all-shared-memory network (still used for the big buckets) was bound by shared-memory wavefronts.
template <int E, int THREADS = 256>
__device__ __forceinline__ void bitonic_sort_regs(const uint64_t* __restrict__ keys, int n, uint32_t* __restrict__ out,
                                                  uint64_t* s)
{
    const int t = threadIdx.x;
    uint64_t v[E];
#pragma unroll
    for (int e = 0; e < E; ++e) v[e] = t * E + e < n ? keys[t * E + e] : kKeyInf;
    constexpr int n2 = THREADS * E;
#pragma unroll 1
    for (int k = 2; k <= n2; k <<= 1) {
#pragma unroll 1
        for (int j = k >> 1; j >= E; j >>= 1) {             // strides across threads
            if (j < 32 * E) {
                const int lm = j / E;
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    const int i = t * E + e;
                    const uint64_t o = __shfl_xor_sync(0xffffffffu, v[e], lm);
                    const bool keep_min = ((i & j) == 0) == ((i & k) == 0);
                    v[e] = keep_min ? min(v[e], o) : max(v[e], o);
                }
            } else {
                // key i = t E + e sits at s[e THREADS + t]: a warp's stores are contiguous, and so are its loads of the
                // partners i ^ j = (t ^ j / E) E + e (j / E >= 32 flips a bit above the lane index): no bank conflicts
#pragma unroll
                for (int e = 0; e < E; ++e) s[e * THREADS + t] = v[e];
                __syncthreads();
                const int tp = t ^ (j / E);
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    const int i = t * E + e;
                    const uint64_t o = s[e * THREADS + tp];
                    const bool keep_min = ((i & j) == 0) == ((i & k) == 0);
                    v[e] = keep_min ? min(v[e], o) : max(v[e], o);
                }
                __syncthreads();
            }
        }
#pragma unroll
        for (int j = E / 2; j > 0; j >>= 1) {               // strides inside a thread: compile-time register indices
            if (j < k) {
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    if ((e & j) == 0) {
                        const int i = t * E + e;
                        const uint64_t a = v[e], b = v[e | j];
                        if ((a > b) == ((i & k) == 0)) { v[e] = b; v[e | j] = a; }
                    }
                }
            }
        }
    }
#pragma unroll
    for (int e = 0; e < E; ++e)
        if (t * E + e < n) out[t * E + e] = (uint32_t)v[e];
}

// LSD radix sort of one bucket of up to 1,024 x E keys in shared memory (1,024 threads), for the buckets above kSmallBucket keys:
// a bitonic network does O(n log^2 n) 64-bit compare-exchanges (config 4: 0.51 ms for 1,689 buckets of 2,049..6,518 keys),
// four 8-bit passes over the DEPTH half of the key do O(n).  Warp w owns the keys [32 E w, 32 E (w + 1)), key (round e, lane)
// at 32 E w + 32 e + lane, so "earlier" means (warp, round, lane) and a stable rank is
//     keys of smaller digits  +  same digit in earlier warps  +  same digit earlier in this warp,
// the last from per-warp digit counters advanced round by round (eight ballots group the lanes of a digit), the second
// from a column scan of those counters, the first from a scan over the 256 digit totals.  A pass in which every real key
// has the same digit is skipped (the sign / exponent byte of the depths of one tile, usually).  Equal depths are then ordered
// by Gaussian id (the low half of the key) in a last step: each key of a run of equal depths counts the smaller ids of its run.
constexpr int kRadixWarps = 32;
template <int E>
__device__ __forceinline__ void radix_sort_bucket(const uint64_t* __restrict__ keys, const int n, uint32_t* __restrict__ out,
                                                  uint64_t* s, uint32_t* cnt)
{
    __shared__ uint32_t base[256], wsum[8];
    const int t = threadIdx.x, lane = t & 31, w = t >> 5;
    const uint32_t lt = (1u << lane) - 1u;
    constexpr int n2 = kRadixWarps * 32 * E;
    const int pad = n2 - n;
    uint32_t* wc = cnt + w * 256;
    uint64_t v[E];
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int i = w * 32 * E + e * 32 + lane;
        v[e] = i < n ? keys[i] : kKeyInf;
    }
#pragma unroll 1
    for (int shift = 32; shift < 64; shift += 8) {
        for (int i = t; i < kRadixWarps * 256; i += kRadixWarps * 32) cnt[i] = 0u;
        __syncthreads();
        uint32_t rank[E];
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const uint32_t d = (uint32_t)(v[e] >> shift) & 255u;
            uint32_t peers = 0xffffffffu;             // lanes with the same digit: eight ballots (MATCH.ANY is far slower)
#pragma unroll
            for (int b = 0; b < 8; ++b) {
                const bool bit = (d >> b) & 1u;
                const uint32_t bal = __ballot_sync(0xffffffffu, bit);
                peers &= bit ? bal : ~bal;
            }
            const uint32_t pre = wc[d];
            __syncwarp();
            if (lane == __ffs(peers) - 1) wc[d] = pre + __popc(peers);
            __syncwarp();
            rank[e] = pre + __popc(peers & lt);
        }
        __syncthreads();
        // column scan over the warps (thread = digit), then the scan over the digits
        uint32_t tot = 0u, incl = 0u;
        if (t < 256) {
#pragma unroll 4
            for (int ww = 0; ww < kRadixWarps; ++ww) {
                const uint32_t x = cnt[ww * 256 + t];
                cnt[ww * 256 + t] = tot;
                tot += x;
            }
            incl = tot;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += y; }
            if (lane == 31) wsum[w] = incl;
        }
        const int same = __syncthreads_or(t < 256 && (int)tot - (t == 255 ? pad : 0) == n);
        if (same) continue;                     // every real key has this digit: the pass would move nothing
        if (t < 256) {
            uint32_t off = 0u;
            for (int ww = 0; ww < w; ++ww) off += wsum[ww];
            base[t] = off + incl - tot;
        }
        __syncthreads();
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const uint32_t d = (uint32_t)(v[e] >> shift) & 255u;
            s[base[d] + wc[d] + rank[e]] = v[e];
        }
        __syncthreads();
#pragma unroll
        for (int e = 0; e < E; ++e) v[e] = s[w * 32 * E + e * 32 + lane];
        __syncthreads();
    }
#pragma unroll
    for (int e = 0; e < E; ++e) s[w * 32 * E + e * 32 + lane] = v[e];
    __syncthreads();
    // equal depths by ascending id
#pragma unroll 1
    for (int e = 0; e < E; ++e) {
        const int i = w * 32 * E + e * 32 + lane;
        if (i >= n) continue;
        const uint64_t key = s[i];
        const uint32_t dep = (uint32_t)(key >> 32), id = (uint32_t)key;
        const bool tl = i > 0 && (uint32_t)(s[i - 1] >> 32) == dep, tr = i + 1 < n && (uint32_t)(s[i + 1] >> 32) == dep;
        int pos = i;
        if (tl || tr) {
            int a = i;
            while (a > 0 && (uint32_t)(s[a - 1] >> 32) == dep) --a;
            int r = 0;
            for (int j = a; j < n && (uint32_t)(s[j] >> 32) == dep; ++j) r += (uint32_t)s[j] < id;
            pos = a + r;
        }
        out[pos] = id;
    }
}

// One CTA per tile.  BIG = false handles buckets of <= kSmallBucket keys (several CTAs per SM), BIG = true the rest:
// up to kBigBucket keys in one shared-memory run; beyond that, runs of kBigBucket keys are sorted one by one and every
// key is then ranked against the other runs by binary search (keys are unique, so ranks are a permutation).
template <bool BIG>
__device__ __forceinline__ void tile_sort_one(const int tile, const int capacity, const int32_t* __restrict__ tile_range,
                                              uint64_t* __restrict__ keys, uint64_t* __restrict__ scratch,
                                              uint32_t* __restrict__ isect_gauss, uint64_t* skeys)
{
    const int start = tile_range[2 * tile];
    const int n = min(tile_range[2 * tile + 1], capacity) - start;      // capacity: see qr_bin_sort (M as an upper bound)
    if (BIG ? (n <= kSmallBucket) : (n <= 0 || n > kSmallBucket)) return;
    constexpr int kRun = BIG ? kBigBucket : kSmallBucket;
    if (!BIG && n > 128) {                      // 256 threads, keys in registers
        if (n <= 256) bitonic_sort_regs<1>(keys + start, n, isect_gauss + start, skeys);
        else if (n <= 512) bitonic_sort_regs<2>(keys + start, n, isect_gauss + start, skeys);
        else if (n <= 1024) bitonic_sort_regs<4>(keys + start, n, isect_gauss + start, skeys);
        else bitonic_sort_regs<8>(keys + start, n, isect_gauss + start, skeys);
        return;
    }
    if (BIG && n <= kRun) {                     // 1,024 threads, 4 / 8 / 16 keys per thread: radix sort in shared memory
        uint32_t* cnt = reinterpret_cast<uint32_t*>(skeys + kBigBucket);
        if (n <= 4096) radix_sort_bucket<4>(keys + start, n, isect_gauss + start, skeys, cnt);
        else radix_sort_bucket<8>(keys + start, n, isect_gauss + start, skeys, cnt);
        __syncthreads();
        return;
    }
    if (n <= kRun) {
        int n2 = 32;
        while (n2 < n) n2 <<= 1;
        for (int i = threadIdx.x; i < n2; i += blockDim.x) skeys[i] = i < n ? keys[start + i] : kKeyInf;
        __syncthreads();
        bitonic_sort_smem(skeys, n2);
        for (int i = threadIdx.x; i < n; i += blockDim.x) isect_gauss[start + i] = (uint32_t)skeys[i];
        __syncthreads();
        return;
    }
    if (BIG) {
        const int nruns = (n + kRun - 1) / kRun;
        for (int r = 0; r < nruns; ++r) {                        // sort each run, back into keys
            const int r0 = r * kRun, rn = min(kRun, n - r0);
            for (int i = threadIdx.x; i < kRun; i += blockDim.x) skeys[i] = i < rn ? keys[start + r0 + i] : kKeyInf;
            __syncthreads();
            bitonic_sort_smem(skeys, kRun);
            for (int i = threadIdx.x; i < rn; i += blockDim.x) keys[start + r0 + i] = skeys[i];
            __syncthreads();
        }
        __threadfence_block();
        __syncthreads();
        for (int i = threadIdx.x; i < n; i += blockDim.x) {      // rank = own index in its run + keys below it elsewhere
            const uint64_t key = keys[start + i];
            const int own = i / kRun;
            int rank = i - own * kRun;
            for (int r = 0; r < nruns; ++r) {
                if (r == own) continue;
                const uint64_t* run = keys + start + r * kRun;
                int lo = 0, hi = min(kRun, n - r * kRun);
                while (lo < hi) {
                    const int mid = (lo + hi) >> 1;
                    if (run[mid] < key) lo = mid + 1; else hi = mid;
                }
                rank += lo;
            }
            scratch[start + rank] = key;
        }
        __syncthreads();
        for (int i = threadIdx.x; i < n; i += blockDim.x) isect_gauss[start + i] = (uint32_t)scratch[start + i];
        __syncthreads();
    }
}

// One CTA per tile in both kernels (a CTA whose bucket belongs to the other kernel returns at once); two CTAs of the
// big kernel (96 KB of shared memory each) fit an SM.
template <bool BIG>
__global__ void __launch_bounds__(BIG ? 1024 : 256)
tile_sort_kernel(const int32_t* __restrict__ tile_range, int32_t T, int32_t capacity, uint64_t* __restrict__ keys,
                 uint64_t* __restrict__ scratch, uint32_t* __restrict__ isect_gauss)
{
    extern __shared__ __align__(16) uint64_t skeys[];
    for (int tile = blockIdx.x; tile < T; tile += gridDim.x) tile_sort_one<BIG>(tile, capacity, tile_range, keys, scratch, isect_gauss, skeys);
}

// inclusive prefix sum of N uint32 counts into uint64 (used by qr_bin_count and by qr_devoxelize); sums: scan_blocks(N) uint64
int64_t scan_blocks(int64_t N) { return N > 0 ? (N + kScanChunk - 1) / kScanChunk : 1; }
int launch_inclusive_scan_u32(const uint32_t* in, int64_t N, uint64_t* out, uint64_t* sums, cudaStream_t st)
{
    const unsigned nb = (unsigned)scan_blocks(N);
    scan_reduce_kernel<<<nb, kScanThreads, 0, st>>>(in, N, sums);
    QR_LAUNCH_OK("scan_reduce_kernel");
    scan_sums_kernel<<<1, kScanThreads, 0, st>>>(sums, (int64_t)nb);
    QR_LAUNCH_OK("scan_sums_kernel");
    scan_apply_kernel<<<nb, kScanThreads, 0, st>>>(in, N, sums, out);
    QR_LAUNCH_OK("scan_apply_kernel");
    return QR_OK;
}

struct BinLayout {
    size_t keys, scratch, counter, sums, total;
    int64_t nblocks_scan;
};

static BinLayout bin_layout(int64_t N, int64_t M, int32_t T)
{
    BinLayout L;
    const size_t m = (size_t)(M > 0 ? M : 1);
    const size_t t = (size_t)(T > 0 ? T : 1);
    L.nblocks_scan = (N + kScanChunk - 1) / kScanChunk;
    if (L.nblocks_scan < 1) L.nblocks_scan = 1;
    size_t o = 0;
    L.sums = o;    o = align_up(o + (size_t)L.nblocks_scan * 8, 256);      // first: qr_bin_count knows neither M nor T
    L.keys = o;    o = align_up(o + m * 8, 256);
    L.scratch = o; o = align_up(o + m * 8, 256);
    L.counter = o; o = align_up(o + t * kSubBuckets * 4, 256);
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
    if (ws_bytes < L.keys)
        return fail(QR_ERR_WORKSPACE_TOO_SMALL, "qr_bin_count: workspace %zu < %zu bytes", ws_bytes, L.keys);
    cudaStream_t st = (cudaStream_t)stream;
    uint64_t* sums = reinterpret_cast<uint64_t*>(static_cast<char*>(ws) + L.sums);
    if (int rc = launch_inclusive_scan_u32(tiles_touched, N, offsets, sums, st)) return rc;
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
        if (ws && ws_bytes >= 8) QR_CUDA_OK(cudaMemsetAsync(ws, 0, 8, st));      // intersections found (N == 0: none; M == 0: not counted)
        return QR_OK;
    }
    (void)offsets;                              // the bucketed sort finds its own offsets (kept in the ABI; may be NULL)
    if (!depth || !tile_rect || !isect_gauss || !ws)
        return fail(QR_ERR_NULL_POINTER, "qr_bin_sort: NULL array");
    if (!aligned16(tile_rect) || !aligned16(ws)) return fail(QR_ERR_MISALIGNED, "qr_bin_sort: tile_rect / ws alignment");
    const BinLayout L = bin_layout(N, M, T);
    if (ws_bytes < L.total)
        return fail(QR_ERR_WORKSPACE_TOO_SMALL, "qr_bin_sort: workspace %zu < %zu bytes", ws_bytes, L.total);
    char* w = static_cast<char*>(ws);
    uint64_t* keys = reinterpret_cast<uint64_t*>(w + L.keys);
    uint64_t* scratch = reinterpret_cast<uint64_t*>(w + L.scratch);
    uint32_t* counter = reinterpret_cast<uint32_t*>(w + L.counter);
    const int4* rects = reinterpret_cast<const int4*>(tile_rect);
    const unsigned nbg = (unsigned)((N + 255) / 256);

    static bool attr_set = false;
    if (!attr_set) {
        QR_CUDA_OK(cudaFuncSetAttribute(tile_sort_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kBigSmem));
        attr_set = true;
    }
    QR_CUDA_OK(cudaMemsetAsync(counter, 0, sizeof(uint32_t) * (size_t)T * kSubBuckets, st));
    tile_bucket_kernel<false><<<nbg, 256, 0, st>>>(N, k.tiles_x, depth, rects, counter, keys, (uint32_t)M);
    QR_LAUNCH_OK("tile_bucket_kernel<count>");
    tile_scan_kernel<<<1, 1024, 0, st>>>(counter, T, tile_range, (uint32_t)M, reinterpret_cast<int64_t*>(w + L.sums));
    QR_LAUNCH_OK("tile_scan_kernel");
    tile_bucket_kernel<true><<<nbg, 256, 0, st>>>(N, k.tiles_x, depth, rects, counter, keys, (uint32_t)M);
    QR_LAUNCH_OK("tile_bucket_kernel<scatter>");
    tile_sort_kernel<false><<<(unsigned)T, 256, kSmallBucket * sizeof(uint64_t), st>>>(tile_range, T, (int32_t)M, keys, scratch, isect_gauss);
    QR_LAUNCH_OK("tile_sort_kernel<small>");
    const int sms = sm_count();
    (void)sms;
    tile_sort_kernel<true><<<(unsigned)T, 1024, kBigSmem, st>>>(tile_range, T, (int32_t)M, keys, scratch, isect_gauss);
    QR_LAUNCH_OK("tile_sort_kernel<big>");
    return QR_OK;
}

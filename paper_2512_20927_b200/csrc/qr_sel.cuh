// qr_sel.cuh -- "selection lists": what the transmittance walk (qr_walk.cu) hands to the two tensor-core contractions,
// the forward blend (qr_blend_mma.cu) and the backward scatter (qr_backward_mma.cu).
//
// The unit is the 16x8-pixel half tile (128 pixels = the M extent of the forward MMA and the K extent of the backward
// one).  For every half tile the lists hold
//   hdr[16]           n[0..3] = entries in each of the four lists, U = number of distinct selected Gaussians (the
//                     "union": the columns of the weight matrix W[128 px, U]), flags; then the walk's work counters,
//                     read only by bench.py's untimed statistics: [6] tile-list entries consumed before every pixel
//                     had stopped, [7] (entry, warp) pairs that survived the culling test (x 32 = alpha' evaluations),
//                     [8] SM clock cycles the half tile's CTA took
//   uid[U]            union column -> Gaussian id (numbered in order of first selection, any order: both contractions
//                     sum over the columns)
//   ent[4][32 K]      one 8-byte entry per selection {weight bits, column << 15 | slot << 7 | pixel}: the NORMALISED
//                     weight w^Q / (1 - T^Q) (Algorithm 1 lines 8 and 20), the column of the
//                     selected Gaussian, the slot of the selection in its pixel's record (depth order) and the pixel's
//                     row-major index inside the half tile.  List q is written by warp q of the walk CTA; lists 0, 1
//                     only hold pixels 0..63 and lists 2, 3 pixels 64..127 (the two W half buffers of the backward).
// Capacities are exact upper bounds (a pixel selects at most K Gaussians), so nothing here can overflow.
#pragma once
#include "qr_common.cuh"

namespace qr {

constexpr int kHalfPx = 128;
constexpr int kSelLists = 4;
constexpr int kHdrWords = 16;

__host__ __device__ __forceinline__ uint32_t sel_pack(int col, int slot, int pixel)
{
    return ((uint32_t)col << 15) | ((uint32_t)slot << 7) | (uint32_t)pixel;
}
__host__ __device__ __forceinline__ int sel_col(uint32_t y) { return (int)(y >> 15); }
__host__ __device__ __forceinline__ int sel_slot(uint32_t y) { return (int)((y >> 7) & 0xFFu); }
__host__ __device__ __forceinline__ int sel_pixel(uint32_t y) { return (int)(y & 127u); }

struct SelLists {
    int32_t* hdr = nullptr;     // [half tiles][kHdrWords]
    int32_t* uid = nullptr;     // [half tiles][ucap]
    uint2* ent = nullptr;       // [half tiles][kSelLists][qcap]
    int32_t ucap = 0, qcap = 0; // 128 K, 32 K
    int32_t* stamp = nullptr;   // [8] magic, width, height, K, low / high word of the sel_idx pointer they describe
    int32_t* ctrl = nullptr;    // [kCtrlWords] [0] the walk's half-tile ticket, [1] the blend's; zeroed per frame
    int32_t* flags = nullptr;   // [half tiles] directly behind ctrl: 1 = the half tile's lists are complete (released)
};
constexpr int kCtrlWords = 64;
// ctrl[8..15] as four uint64: kernel time stamps of the last frame (%globaltimer, ns), read by bench.py's untimed
// statistics only: [0] ~first walk CTA start (stored as ~t so that atomicMax finds the minimum), [1] last walk CTA end,
// [2] ~first blend CTA start, [3] last blend CTA end
__device__ __forceinline__ void stamp_time(int32_t* ctrl, int slot, bool is_start)
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    atomicMax(reinterpret_cast<unsigned long long*>(ctrl + 8) + slot, is_start ? ~t : t);
}

struct SelLayout {
    size_t stamp, ctrl, hdr, uid, ent, total;
    int32_t ucap, qcap;
};
inline SelLayout sel_layout(const Cam& cam, int K, size_t base = 0)
{
    const size_t nh = (size_t)cam.tiles_x * cam.tiles_y * 2;
    SelLayout L;
    L.ucap = kHalfPx * K;
    L.qcap = 32 * K;
    size_t o = base;
    L.stamp = o; o = align_up(o + 64, 256);
    L.ctrl = o;  o = align_up(o + ((size_t)kCtrlWords + nh) * 4, 256);
    L.hdr = o;   o = align_up(o + nh * kHdrWords * 4, 256);
    L.uid = o;   o = align_up(o + nh * (size_t)L.ucap * 4, 256);
    L.ent = o;   o = align_up(o + nh * kSelLists * (size_t)L.qcap * 8, 256);
    L.total = o;
    return L;
}
inline SelLists sel_view(const SelLayout& L, void* ws)
{
    char* w = static_cast<char*>(ws);
    SelLists s;
    s.stamp = reinterpret_cast<int32_t*>(w + L.stamp);
    s.ctrl = reinterpret_cast<int32_t*>(w + L.ctrl);
    s.flags = s.ctrl + kCtrlWords;
    s.hdr = reinterpret_cast<int32_t*>(w + L.hdr);
    s.uid = reinterpret_cast<int32_t*>(w + L.uid);
    s.ent = reinterpret_cast<uint2*>(w + L.ent);
    s.ucap = L.ucap; s.qcap = L.qcap;
    return s;
}
constexpr int32_t kSelMagic = 0x51524c31;   // "QRL1"

// Common layout of the qr_forward and the qr_backward workspace (fp32 features, D % 128 == 0: the tcgen05 paths), so that
// qr_backward_lists and qr_backward_clear can be handed either one:
//   [0, 256)      scratch words of the owning call (qr_backward: [0] half tiles left to the FFMA kernel)
//   [256, ...)    selection lists: stamp, tickets + release flags, headers, union ids, entries
//   then          qr_backward_clear's de-duplication cache (kSeenCells ints)
constexpr int kSeenCells = 1 << 20;
struct WsLayout { SelLayout sel; size_t seen, total; };
inline WsLayout ws_layout(const Cam& cam, int K)
{
    WsLayout L;
    L.sel = sel_layout(cam, K, 256);
    L.seen = L.sel.total;
    L.total = align_up(L.seen + (size_t)kSeenCells * 4, 256);
    return L;
}
// device-side check that lists belong to this camera and K (anything else: the kernel leaves without touching memory)
__device__ __forceinline__ bool sel_stamp_ok(const int32_t* stamp, const Cam& cam, int K)
{
    return stamp[0] == kSelMagic && stamp[1] == cam.width && stamp[2] == cam.height && stamp[3] == K;
}

// qr_walk.cu
struct WalkParams2 {
    Cam cam;
    int32_t K;
    const float2* mean2d;
    const float4* conic_opac;
    const uint32_t* isect;
    const int2* tile_range;
    int32_t* n_sel;
    float* resid;
    int32_t* sel_idx;
    float* sel_w;
    SelLists sl;
    int32_t batch_n = 0;    // qr_forward_batch: ids in isect are virtual (view * N + Gaussian); 0 = single view
    int32_t view_h = 0;     //                   rows per view of the tall image; 0 = single view
    float2* stats = nullptr;   // stratified-K: per pixel (mu, sigma) of the dense transmittance values (pass 1 writes, pass 2 reads)
    float t_min = 0.0f, z_max = 2.0f;
};
// Several K in ONE walk (second half): staging, culling, alpha' and the dense transmittance T are shared,
// every K has its own boundaries, T^Q, records and selection lists.
constexpr int kMaxMultiK = 4;
struct WalkParamsMulti {
    Cam cam;
    int32_t nK;
    int32_t K[kMaxMultiK];
    const float2* mean2d;
    const float4* conic_opac;
    const uint32_t* isect;
    const int2* tile_range;
    int32_t* n_sel[kMaxMultiK];
    float* resid[kMaxMultiK];
    int32_t* sel_idx[kMaxMultiK];
    float* sel_w[kMaxMultiK];
    SelLists sl[kMaxMultiK];
};
int launch_walk2_multi(const WalkParamsMulti& p, cudaStream_t st);

int launch_walk2(const WalkParams2& p, cudaStream_t st);
int launch_walk2_stratified(const WalkParams2& p, cudaStream_t st);
// dense comparator: entries = every blended (Gaussian, pixel) pair with its weight T alpha' (p.t_min: stop rule R7; p.resid receives
// the final transmittance; p.K = list capacity in entries per pixel; no records: p.sel_idx / p.sel_w / p.n_sel unused)
int launch_walk2_dense(const WalkParams2& p, cudaStream_t st);

}  // namespace qr

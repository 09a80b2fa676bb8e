/*
 * qr.h -- C ABI of libqr: the data-parallel hot path of Quantile Rendering (Q-Render) on B200 (sm_100a).
 *
 * The calls split  f~^Q = QuantileRender(G, F, K, I)  (Algorithm 1 at PAPER.md:129-158) at the
 * stage boundaries of the 3D-GS pipeline the paper builds on ("(1) tiling strategy; (2) splatting
 * algorithm [EWA]; (3) volume rendering"):
 *
 *   qr_preprocess      EWA projection of means / covariances to 2D conics, tile rectangles, depth
 *   qr_bin_count       prefix sum of tiles touched -> M = number of (Gaussian, tile) intersections
 *   qr_bin_sort        tile-intersection duplication, (tile, depth) radix sort, per-tile ranges
 *   qr_forward         per-pixel transmittance walk, quantile selection, K-sparse feature accumulation
 *   qr_backward        dL/dfeature scatter-add to the selected Gaussians (qr_backward_clear re-zeroes those rows)
 *   qr_dense_forward   Eq. 1 dense volume rendering of the same features (in-run comparator)
 *
 * Conventions the paper leaves to "[3D-GS]" are fixed in DESIGN.md ("Readings", R1-R15).
 *
 * Pointers.  Every pointer is a DEVICE pointer owned by the caller unless marked HOST.  The library allocates
 * nothing persistent: scratch comes from caller-provided workspaces sized by the *_workspace_bytes() calls.
 * Inputs are never modified.  Device pointers must be 16-byte aligned.
 * Streams.   `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Every call only
 * enqueues work on `stream` and returns, except qr_bin_count, which also waits for `stream` to deliver M.
 * Errors.    Return value 0 = QR_OK, negative = qr_status.  No call throws, aborts or prints; on error nothing
 * is enqueued and qr_last_error() gives a thread-local HOST string.  Degenerate but legal inputs (N = 0, M = 0,
 * a pixel with no Gaussian) are not errors.
 */
#ifndef QR_H_
#define QR_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define QR_VERSION 200       /* major*10000 + minor*100 + patch */
#define QR_TILE 16           /* tile edge in pixels (3D-GS convention) */
#define QR_MAX_K 256         /* largest K qr_forward / qr_backward accept */
#define QR_TOPK_MAX_K 64      /* largest K qr_topk_forward accepts (the paper sweeps 5..50) */
#define QR_MAX_BATCH 16       /* views per batched call (the paper trains on 4 viewpoints per step) */
#define QR_MAX_MASKS 2048     /* masks per frame qr_mask_loss accepts */
#define QR_REDUCE_MEAN 0
#define QR_REDUCE_MAX 1
#define QR_MAX_D 512         /* largest feature width ("up to 512-D") */

typedef enum {
    QR_OK = 0,
    QR_ERR_INVALID_ARG = -1,          /* size / range violation (K < 1, width < 1, ...) */
    QR_ERR_NULL_POINTER = -2,
    QR_ERR_UNSUPPORTED = -3,          /* K > QR_MAX_K, D > QR_MAX_D, fp16 with D % 8 != 0, D % 4 != 0 with D > 128 */
    QR_ERR_WORKSPACE_TOO_SMALL = -4,
    QR_ERR_CAPACITY = -5,             /* M does not fit the arithmetic of the sort (M >= 2^31) */
    QR_ERR_CUDA = -6,                 /* a CUDA runtime call failed; qr_last_error() has its message */
    QR_ERR_MISALIGNED = -7
} qr_status;

typedef enum { QR_F32 = 0, QR_F16 = 1 } qr_dtype;

/* HOST struct.  Pinhole camera; pixel (x, y) samples the image plane at (x + 0.5, y + 0.5) (reading R5). */
typedef struct {
    int32_t width, height;   /* >= 1 */
    float fx, fy, cx, cy;    /* pixels */
    float znear;             /* > 0; a Gaussian whose camera-space z <= znear is culled */
    float world_to_cam[12];  /* row-major 3x4 [R|t], R orthonormal; camera looks along +z, y down */
} qr_camera;

int qr_version(void);
const char* qr_last_error(void);   /* HOST string, thread-local, valid until the next failing call on this thread */

/* Kernels this process has launched through the library so far (every launch is counted where it is issued;
 * memsets are not kernels and are not counted).  bench.py reports the difference over its timed region. */
long long qr_launch_count(void);

/* Number of tiles of a camera: ceil(width/16) * ceil(height/16).  Returns 0 for a NULL or zero-area camera. */
int32_t qr_num_tiles(const qr_camera* cam);

/*
 * qr_preprocess -- PAPER.md:79 (Sigma = R S S^T R^T), PAPER.md:80/:124 (EWA splatting "following [3D-GS]"),
 * SPEC.md:130-138, :163-168.  One thread per Gaussian, fp32, operation order fixed in DESIGN.md
 * ("fp32 decision arithmetic") so that `depth` -- the sort key -- is reproducible bit for bit.
 *   in : means[N,3], scales[N,3] (> 0), quats[N,4] (w,x,y,z; unit), opac[N] in (0,1)
 *   out: mean2d[N,2] pixel coordinates; conic_opac[N,4] = (a, b, c) of cov2d^-1 and the opacity;
 *        depth[N] camera-space z (written for every Gaussian); tile_rect[N,4] = x0,y0,x1,y1 half-open tile
 *        rectangle of the 3-sigma AABB clamped to the tile grid; tiles_touched[N] (0 = culled; all other
 *        outputs of a culled Gaussian except depth are 0).
 * N = 0 is legal (nothing enqueued).
 */
int qr_preprocess(const qr_camera* cam, int64_t N,
                  const float* means, const float* scales, const float* quats, const float* opac,
                  float* mean2d, float* conic_opac, float* depth,
                  int32_t* tile_rect, uint32_t* tiles_touched, void* stream);

/*
 * qr_bin_count -- inclusive prefix sum of tiles_touched ("(1) tiling strategy").
 *   out: offsets[N] (uint64, inclusive scan); *M_host (HOST) = offsets[N-1] = number of intersections.
 * Performs the one device->host read of the path and synchronises `stream`.
 */
size_t qr_bin_workspace_bytes(int64_t N, int64_t M_capacity, int32_t num_tiles);
int qr_bin_count(int64_t N, const uint32_t* tiles_touched, uint64_t* offsets, int64_t* M_host,
                 void* ws, size_t ws_bytes, void* stream);

/*
 * qr_bin_sort -- duplication + sort + ranges ("ordered sequence of indices"; SPEC.md:139-147,
 * :167-168; reading R6: order = ascending depth, ties by ascending Gaussian index).
 * Each un-culled Gaussian emits one entry per tile of its rectangle.  One most-significant-digit radix pass over the
 * tile field (count, scan, scatter: a counting sort with one bucket per tile) is followed by a sort of every bucket
 * on its 64-bit (IEEE bits of depth << 32 | Gaussian id) keys; the keys are unique, so the result does not depend on
 * the order the buckets were filled in.
 *   in : depth[N], tile_rect[N,4]; M = capacity of isect_gauss: the exact count from qr_bin_count, or any upper
 *        bound (e.g. from the previous frame) when the caller wants no host synchronisation; offsets is unused by
 *        this implementation and may be NULL.
 *   out: isect_gauss[M] Gaussian ids sorted by (tile, depth, id); tile_range[T,2] = [start, end) of tile t in
 *        isect_gauss (empty tile: start == end == number of intersections in tiles < t);
 *        ((int64_t*)ws)[0] = number of intersections found.  If it exceeds M the lists are truncated at M entries
 *        (ranges clamped, nothing is written out of bounds): call again with a larger M.
 * ws must hold qr_bin_workspace_bytes(N, M, T) bytes.  M = 0 is legal (ranges are all [0,0)).
 */
int qr_bin_sort(const qr_camera* cam, int64_t N, int64_t M,
                const float* depth, const int32_t* tile_rect, const uint64_t* offsets,
                uint32_t* isect_gauss, int32_t* tile_range, void* ws, size_t ws_bytes, void* stream);

/*
 * qr_forward -- Algorithm 1 for every pixel, then f~^Q = f^Q / (1 - T^Q).
 * Inclusion rule R4: Gaussian i is in pixel p's list I iff power = -1/2 d^T conic d is in [-4.5, 0] and
 * alpha' = min(0.99, opacity * exp(power)) >= 1/255.  Strict comparisons against 1 - (k+1)/(K+1) in fp32 (R2, R3).
 *   in : mean2d, conic_opac (qr_preprocess); isect_gauss, tile_range (qr_bin_sort);
 *        features[N,D] row-major, fp32 or fp16 (feat_dtype); fp16 is widened exactly, accumulation is fp32.
 *   out: out_map[H,W,D] fp32 (HWC; 0 where nothing is selected, R8)
 *        sel_idx[H,W,K] int32 selected Gaussian ids in depth order; only slots s < n_sel[p] are part of the result:
 *        sel_w[H,W,K]   fp32 normalised weights w^Q / (1 - T^Q)       the others are left as the caller passed them
 *        n_sel[H,W]     int32 number selected (<= K)                  (writing -1 / 0 there would be two thirds of the
 *        resid_TQ[H,W]  fp32 T^Q after the walk (1 where nothing is selected)     records' traffic, for no reader)
 * out_map may be NULL on the tcgen05 path (see below): selection only -- the walk, the records and the selection
 * lists, no blend, no map (what qr_pooled_loss needs).
 * K in [1, QR_MAX_K]; D in [1, QR_MAX_D]; D % 4 == 0 unless D <= 128; fp16 needs D % 8 == 0.
 * ws must hold qr_forward_workspace_bytes(cam, K, D) bytes; every pointer must be non-NULL.  For fp32 or fp16 features with
 * D % 32 == 0, or D < 32 with D % 4 == 0 (the tcgen05 path: the contractions run on whole 128-channel tiles and let TMA pad the
 * loads with zeros and clip the stores; fp16 additionally D % 8 == 0) the call leaves in ws, per 16x8-pixel half tile, the numbered union of selected
 * Gaussians and the selection as (weight, column, pixel) entries; qr_backward_lists and qr_backward_clear accept that
 * workspace as it is, until the next call that writes it.
 */
size_t qr_forward_workspace_bytes(const qr_camera* cam, int32_t K, int32_t D);
int qr_forward(const qr_camera* cam, int32_t K, int32_t D, qr_dtype feat_dtype,
               const float* mean2d, const float* conic_opac,
               const uint32_t* isect_gauss, const int32_t* tile_range, const void* features,
               float* out_map, int32_t* sel_idx, float* sel_w, int32_t* n_sel, float* resid_TQ,
               void* ws, size_t ws_bytes, void* stream);

/*
 * qr_forward_stats -- work counters of the last qr_forward that took the tcgen05 path (the shapes named at qr_forward), summed over
 * the half-tile headers it left in its workspace ("the bench must report this count"):
 *   stats[0] selections (sum of n_sel)            stats[1] sum over half tiles of U_ht (distinct Gaussians selected)
 *   stats[2] tile-list entries consumed before every pixel of the half tile had stopped
 *   stats[3] (entry, pixel) alpha' evaluations of the walk (32 x the (entry, warp) pairs that survived the culling test)
 *   stats[4] SM clock cycles summed over the walk's half tiles      stats[5] half tiles with U_ht > 64 (two+ MMA rounds)
 * stats is a DEVICE array of 8 int64; the call enqueues a memset and one small kernel on `stream`.
 */
int qr_forward_stats(const qr_camera* cam, int32_t K, const void* fwd_ws, size_t fwd_ws_bytes, int64_t* stats, void* stream);

/*
 * qr_backward -- PAPER.md:37, :210.  The selection is piecewise constant in alpha' and the
 * Gaussians are frozen, so the only gradient is
 *     dL/dF[i,:] += sum over pixels p and slots s with sel_idx[p,s] == i of  sel_w[p,s] * dL_dmap[p,:].
 *   in : sel_idx, sel_w, n_sel (from qr_forward), dL_dmap[H,W,D] fp32
 *   out: dL_dfeat[N,D] fp32, ACCUMULATED INTO (the caller zeroes it; rows never selected are left untouched).
 * Summation order over pixels is not fixed (fp32 atomics): results agree to rounding, not bit for bit.
 * ws must hold qr_backward_workspace_bytes(cam, K, D) bytes.  Its contents are scratch: per half tile, the numbered
 * union of selected Gaussians and the selection as (weight, row, pixel) (tcgen05 shapes), and qr_backward_clear's
 * de-duplication cache; for the other shapes qr_backward itself does not touch ws (it may be NULL there).
 */
size_t qr_backward_workspace_bytes(const qr_camera* cam, int32_t K, int32_t D);
int qr_backward(const qr_camera* cam, int32_t K, int32_t D, int64_t N,
                const int32_t* sel_idx, const float* sel_w, const int32_t* n_sel, const float* dL_dmap,
                float* dL_dfeat, void* ws, size_t ws_bytes, void* stream);

/*
 * qr_backward_lists -- the same gradient as qr_backward, computed from the per-half-tile selection lists that the last
 * qr_forward(cam, K, D, ...) left in ITS workspace fwd_ws (see qr_forward), instead of re-deriving the unions
 * from sel_idx / sel_w: one kernel instead of two.  Shapes of the tcgen05 path only (QR_ERR_UNSUPPORTED otherwise).
 * The lists carry a stamp (image size, K) that the kernel checks on the device: a workspace that does not hold the
 * lists of this camera and K makes the call a no-op (dL_dfeat untouched).  fwd_ws is only read.
 */
int qr_backward_lists(const qr_camera* cam, int32_t K, int32_t D, int64_t N, void* fwd_ws, size_t fwd_ws_bytes,
                      const float* dL_dmap, float* dL_dfeat, void* stream);

/*
 * qr_backward_clear -- zero exactly the rows of dL_dfeat that qr_backward over the same selection adds into (the
 * distinct Gaussians selected anywhere in the frame), and nothing else.  A loop that keeps dL_dfeat zero outside
 * those rows (zero it once, then clear after each use) writes ~|S| D floats per step instead of N D
 * (the whole-table zero fill costs more than qr_backward's own traffic).
 *   in : sel_idx, n_sel (from qr_forward); ws / ws_bytes = the workspace AS LEFT BY the last qr_backward call with
 *        the same cam, K, D and selection, or -- after qr_backward_lists -- the forward's workspace (its per-half-tile
 *        unions are reused, a scratch region of it is written).  A workspace whose stamp does not match cam and K is
 *        not trusted: the rows are then found from sel_idx / n_sel.  Ids outside [0, N) are ignored.
 *   out: dL_dfeat rows of selected Gaussians = 0; other rows untouched.
 */
int qr_backward_clear(const qr_camera* cam, int32_t K, int32_t D, int64_t N,
                      const int32_t* sel_idx, const int32_t* n_sel, float* dL_dfeat,
                      void* ws, size_t ws_bytes, void* stream);

/*
 * qr_dense_forward -- Eq. 1: out = sum_i T_i alpha'_i f_i over the same per-pixel lists, not
 * normalised.  Early stop R7: before blending i, T_test = T (1 - alpha'_i); if
 * T_test < t_min stop without blending i.  t_min = 0 is exact Eq. 1.
 *   out: out_map[H,W,D] fp32; final_T[H,W] fp32 transmittance after the last blended Gaussian.
 */
int qr_dense_forward(const qr_camera* cam, int32_t D, qr_dtype feat_dtype, float t_min,
                     const float* mean2d, const float* conic_opac,
                     const uint32_t* isect_gauss, const int32_t* tile_range, const void* features,
                     float* out_map, float* final_T, void* stream);

/*
 * qr_forward_multik -- qr_forward for nK values of K in ONE walk ("multi-K in one walk"; the K sweep of
 * BASELINE.json configs[3]).  Staging, culling, alpha' and the dense transmittance are computed once; every K
 * has its own boundaries, records and selection lists, and its own blend.  For each K the outputs are those of
 * qr_forward(cam, K, ...): identical n_sel, sel_idx, sel_w and resid_TQ; the same map to fp32 summation order; the same
 * selection lists in ws[j] (qr_backward_lists / qr_backward_clear / qr_pooled_loss take ws[j] with K[j]).
 *   Ks: HOST array of nK values in [1, QR_MAX_K], nK in [1, QR_MAX_MULTI_K].
 *   out_map, sel_idx, sel_w, n_sel, resid_TQ, ws: HOST arrays of nK DEVICE pointers (out_map[j] may be NULL: selection only);
 *   ws_bytes[j] >= qr_forward_workspace_bytes(cam, K[j], D); the workspaces must be distinct.
 * Shapes of the tcgen05 path only (QR_ERR_UNSUPPORTED otherwise).
 */
#define QR_MAX_MULTI_K 4
int qr_forward_multik(const qr_camera* cam, int32_t nK, const int32_t* Ks, int32_t D, qr_dtype feat_dtype,
                      const float* mean2d, const float* conic_opac, const uint32_t* isect_gauss, const int32_t* tile_range,
                      const void* features, float* const* out_map, int32_t* const* sel_idx, float* const* sel_w,
                      int32_t* const* n_sel, float* const* resid_TQ, void* const* ws, const size_t* ws_bytes, void* stream);

/*
 * qr_dense_forward_tc -- qr_dense_forward (same definition, same outputs) with the blend on the tensor cores: the walk emits every
 * blended (Gaussian, pixel) pair with its weight T alpha' as selection lists and the tcgen05 contraction of qr_forward renders
 * them, so that Q-Render is compared with a dense renderer built from the same parts.  `cap` = entries per pixel the lists hold
 * (average over each 32-pixel list; 1..QR_MAX_K); half tiles that need more are rendered by qr_dense_forward's FFMA kernel
 * inside the same call.  Shapes of the tcgen05 path only (see qr_forward; QR_ERR_UNSUPPORTED otherwise).  ws must hold
 * qr_dense_workspace_bytes(cam, cap) bytes (scratch).  Results equal qr_dense_forward's to fp32 rounding (summation order).
 */
size_t qr_dense_workspace_bytes(const qr_camera* cam, int32_t cap);
int qr_dense_forward_tc(const qr_camera* cam, int32_t D, qr_dtype feat_dtype, float t_min, int32_t cap,
                        const float* mean2d, const float* conic_opac, const uint32_t* isect_gauss, const int32_t* tile_range,
                        const void* features, float* out_map, float* final_T, void* ws, size_t ws_bytes, void* stream);

/*
 * qr_topk_forward -- the paper's second comparator, top-K render ("top-K sampling ... requires additional
 * complexity to sort values, O(N log K + KC)"; complexity table; "top-K sorts and selects K
 * Gaussians").  The paper gives no procedure; this is the reconstruction of SPEC.md:221-229 (reading R17):
 * dense weights w_i = T_i alpha'_i of Eq. 1 over the pixel's list (same inclusion rule R4 and early stop R7 / t_min as
 * qr_dense_forward), the K largest kept (ties -> the earlier list position), re-blended in depth order with a fresh
 * transmittance T^top, normalised by 1 - T^top like Algorithm 1 line 20; nothing kept -> zero vector, resid = 1.
 *   in : as qr_forward, plus t_min (>= 0; 1e-4 by convention, 0 = weights over the whole list)
 *   out: out_map[H,W,D] fp32; sel_idx / sel_w / n_sel / resid in qr_forward's record format (slots s < n_sel[p] are
 *        written; n_sel[p] = min(K, weighted entries)), so qr_backward accepts them as they are.
 * K in [1, QR_TOPK_MAX_K].  ws must hold qr_topk_workspace_bytes(cam, K, D) bytes (scratch; used for the tcgen05 shapes,
 * where the blend is the same tcgen05 contraction as qr_forward's; may be NULL otherwise).
 */
size_t qr_topk_workspace_bytes(const qr_camera* cam, int32_t K, int32_t D);
int qr_topk_forward(const qr_camera* cam, int32_t K, int32_t D, qr_dtype feat_dtype, float t_min,
                    const float* mean2d, const float* conic_opac,
                    const uint32_t* isect_gauss, const int32_t* tile_range, const void* features,
                    float* out_map, int32_t* sel_idx, float* sel_w, int32_t* n_sel, float* resid,
                    void* ws, size_t ws_bytes, void* stream);

/*
 * qr_forward_stratified -- the paper's stratified-K variant ("we compute the mean and
 * standard deviation of the transmittance values along the depth dimension ... uniformly partition the transmittance interval
 * in the z-score space and then map the samples back"; "two passes along each ray").  DESIGN.md reading R18:
 *   pass 1: per pixel, mu and sigma (population) of the dense transmittance values T_i over its list up to the stop R7 (t_min);
 *   pass 2: Algorithm 1 with the boundaries b_k = clamp(mu + sigma z_k, 0, 1), z_k = z_max (1 - 2 (k+1) / (K+1)), k < K, in
 *           place of 1 - (k+1)/(K+1); the walk ends once T_test < max(b_{K-1}, t_min); sigma == 0 -> Q-Render's boundaries.
 * Inputs and outputs as qr_forward (the records and the workspace's selection lists have the same format: qr_backward,
 * qr_backward_lists and qr_backward_clear accept them); z_max = 2 by convention.  Shapes of the tcgen05 path only
 * (QR_ERR_UNSUPPORTED otherwise).  ws must hold qr_stratified_workspace_bytes(cam, K, D) bytes.
 */
size_t qr_stratified_workspace_bytes(const qr_camera* cam, int32_t K, int32_t D);
int qr_forward_stratified(const qr_camera* cam, int32_t K, int32_t D, qr_dtype feat_dtype, float t_min, float z_max,
                          const float* mean2d, const float* conic_opac,
                          const uint32_t* isect_gauss, const int32_t* tile_range, const void* features,
                          float* out_map, int32_t* sel_idx, float* sel_w, int32_t* n_sel, float* resid_TQ,
                          void* ws, size_t ws_bytes, void* stream);

/*
 * Multi-camera batching ("rendering loss from 4 randomly chosen training viewpoints"): B views
 * of the same Gaussians, same image size (height % 16 == 0), rendered by ONE set of launches and back-propagated into ONE
 * dL_dfeat.  The B tile grids are stacked into one tall grid of B * tiles_y tile rows; everything after the projection works on
 * that tall image as on any other, with two indirections inside the walk: a list entry v = b * N + i ("virtual Gaussian") is
 * looked up in the projected arrays as v and reported (sel_idx, union ids, feature / gradient rows) as i, and alpha' is evaluated
 * in the view's own pixel coordinates -- so every per-view result is what the single-view calls give for that camera.
 *
 *   qr_batch_camera      tall = cams[0] with height B * H: the camera to pass to qr_bin_sort, qr_forward_batch,
 *                        qr_backward / qr_backward_lists / qr_backward_clear and the workspace-size calls.
 *   qr_preprocess_batch  qr_preprocess for cams[0..B) (HOST array) in one launch; every output array has B * N entries, view b
 *                        in [b N, (b+1) N); mean2d / conic_opac / depth are bit-identical to qr_preprocess(cams[b]); tile_rect
 *                        rows are offset by b * tiles_y.  qr_bin_count / qr_bin_sort then take B * N as their N.
 *   qr_forward_batch     qr_forward on the tall image: out_map [B*H, W, D], records [B*H, W, ...]; N = Gaussians per view.
 * Errors as the single-view calls; B outside [1, QR_MAX_BATCH], unequal image sizes or height % 16 != 0: QR_ERR_INVALID_ARG.
 */
int qr_batch_camera(const qr_camera* cams, int32_t B, qr_camera* tall);
int qr_preprocess_batch(const qr_camera* cams, int32_t B, int64_t N,
                        const float* means, const float* scales, const float* quats, const float* opac,
                        float* mean2d, float* conic_opac, float* depth,
                        int32_t* tile_rect, uint32_t* tiles_touched, void* stream);
int qr_forward_batch(const qr_camera* tall, int32_t B, int64_t N, int32_t K, int32_t D, qr_dtype feat_dtype,
                     const float* mean2d, const float* conic_opac,
                     const uint32_t* isect_gauss, const int32_t* tile_range, const void* features,
                     float* out_map, int32_t* sel_idx, float* sel_w, int32_t* n_sel, float* resid_TQ,
                     void* ws, size_t ws_bytes, void* stream);

/*
 * The two neighbours of the path.
 *
 * qr_devoxelize -- PAPER.md:1121-1179 (Listing 3): the 3D network predicts uni_pred[U,C], one row per UNIQUE voxel; Gaussian g
 * was sampled into num_voxels_per_g[g] consecutive voxels, and inverse_indices[v] names the unique voxel of sampled voxel v.
 *   gs_pred[g,:] = REDUCE over the voxels v of g of uni_pred[inverse_indices[v],:],  REDUCE = mean or componentwise max
 * (a Gaussian without voxels gets a zero row).  This is F, the feature table qr_forward reads.  For max, argmax[g,c] receives
 * the first voxel attaining the maximum (-1: none), which qr_devoxelize_backward needs.  The call also leaves the cumulative
 * voxel offsets in ws; qr_devoxelize_backward reads them from the same ws.  C <= 512.  Indices are trusted (out of
 * range is a contract violation).
 * qr_devoxelize_backward -- the adjoint: d_uni[u,:] += sum over voxels v with inverse_indices[v] == u of d_gs[g(v),:] / count
 * (mean) or of d_gs[g(v),c] where v == argmax[g(v),c] (max).  d_gs is dL/dF as qr_backward produces it; d_uni is ACCUMULATED INTO.
 */
size_t qr_devoxelize_workspace_bytes(int64_t G);
int qr_devoxelize(int64_t U, int32_t C, int64_t G, const float* uni_pred, const int64_t* inverse_indices,
                  const uint32_t* num_voxels_per_g, int32_t reduce, float* gs_pred, int32_t* argmax,
                  void* ws, size_t ws_bytes, void* stream);
int qr_devoxelize_backward(int64_t U, int32_t C, int64_t G, const int64_t* inverse_indices, int32_t reduce,
                           const int32_t* argmax, const float* d_gs, float* d_uni,
                           const void* ws, size_t ws_bytes, void* stream);

/*
 * qr_mask_loss -- the training loss of PAPER.md:216-228 (Eq. 2) on a rendered map, and its gradient dL/dmap (the input of
 * qr_backward).  DESIGN.md reading R19 (the printed denominator and the pooling are ambiguous):
 *   pooled_s = mean of map over the pixels p with mask_id[p] == s;  c_j = cos(pooled_s, targets[j]);
 *   L_s = log sum_j exp(c_j) - c_s  (all S targets in the denominator);  L = mean of L_s over masks with pixels and pooled_s != 0.
 *   in : map[H,W,D] fp32, mask_id[H,W] int32 in [0, S) or -1, targets[S,D] fp32 (any non-zero norm)
 *   out: loss[1] (device), loss_per_mask[S] (0 for skipped masks), d_map[H,W,D] = dL/dmap (0 outside every mask)
 * D % 4 == 0, D <= 512, S <= QR_MAX_MASKS.  ws must hold qr_mask_loss_workspace_bytes(S, D) bytes.
 */
size_t qr_mask_loss_workspace_bytes(int32_t S, int32_t D);
int qr_mask_loss(const qr_camera* cam, int32_t D, int32_t S, const float* map, const int32_t* mask_id,
                 const float* targets, float* loss, float* loss_per_mask, float* d_map,
                 void* ws, size_t ws_bytes, void* stream);

/*
 * qr_mask_loss_static -- qr_mask_loss (same inputs, outputs, kernels and arithmetic) for callers that cannot allocate device
 * memory: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The workspace is a
 * file-scope device array of QR_STATIC_SCRATCH_BYTES inside the library (every GPU that loads the library holds it until
 * exit); the call performs no cudaMalloc / cudaFree and calls no allocating library routine (two cudaMemsetAsync, four kernel
 * launches; on its first use per device, one cudaGetSymbolAddress).
 * Limit: qr_mask_loss_workspace_bytes(S, D) <= QR_STATIC_SCRATCH_BYTES, i.e. S <= QR_STATIC_MAX_MASKS = 256 masks at D = 512
 * (more at a smaller D); beyond it QR_ERR_UNSUPPORTED with the sizes in qr_last_error().  Other errors as qr_mask_loss.
 * Every call on a device shares the one array, which keeps the previous call's contents (the call clears what it needs at its
 * start, on `stream`): calls that overlap on the GPU -- two streams, two host threads -- RACE on it; serialise them.
 */
#define QR_STATIC_MAX_MASKS 256
#define QR_STATIC_SCRATCH_BYTES (QR_STATIC_MAX_MASKS * 512 * 4 + 3 * 1024)
int qr_mask_loss_static(const qr_camera* cam, int32_t D, int32_t S, const float* map, const int32_t* mask_id,
                        const float* targets, float* loss, float* loss_per_mask, float* d_map, void* stream);

/*
 * qr_pooled_loss -- qr_mask_loss and qr_backward FUSED with the render path, without the map ("would let
 * qr_forward / qr_backward skip the 629 MB map round-trip").  Rendering is linear in the features and the loss pools the map by
 * a mean per mask, so with A[i,s] = sum over the pixels p of mask s of the normalised weight of Gaussian i at p,
 *     pooled_s = (1 / |m_s|) sum_i A[i,s] F[i,:]      and      dL/dF[i,:] = sum_s A[i,s] g_s     (g_s = dL/dmap on mask s):
 * both directions need only A, which the selection lists of the last qr_forward(cam, K, D, QR_F32, ...) in fwd_ws give per
 * half tile.  Same loss, per-mask losses and gradient as qr_mask_loss on that forward's map followed by qr_backward on its
 * dL/dmap (to rounding), at a fraction of the traffic: neither out_map nor dL/dmap is read or written (call qr_forward with
 * out_map = NULL for a training step).
 *   in : fwd_ws (only read; stamp checked on the device as in qr_backward_lists), features[N,D] fp32, mask_id[H,W], targets[S,D]
 *   out: loss[1], loss_per_mask[S]; dL_dfeat[N,D] ACCUMULATED INTO (may be NULL: loss only)
 * fp32, shapes of the tcgen05 path (see qr_forward), D <= 512.  ws must hold qr_mask_loss_workspace_bytes(S, D) bytes.
 */
int qr_pooled_loss(const qr_camera* cam, int32_t K, int32_t D, int64_t N, void* fwd_ws, size_t fwd_ws_bytes,
                   const float* features, const int32_t* mask_id, int32_t S, const float* targets,
                   float* loss, float* loss_per_mask, float* dL_dfeat, void* ws, size_t ws_bytes, void* stream);

/*
 * qr_sh_colors -- the RGB payload of PAPER.md:940-947 (App. E.6: Q-Render applied to pre-trained 3D-GS models; SURVEY.md 8(f)
 * NEXT-4), reading R20: the view-dependent colour of every Gaussian from its spherical-harmonics coefficients,
 *     colors[i,c] = max(0, 1/2 + sum_k Y_k(dir_i) sh[i,k,c]),   dir_i = unit vector from the camera centre (-R^T t) to means[i],
 * Y_k the real harmonics of degree <= `degree` ordered (l, m = -l..l) with the Condon-Shortley phase kept (degree-1 terms
 * (-y, z, -x) sqrt(3 / (4 pi))).  A Gaussian at the camera centre keeps the constant term only.  colors[N,3] is then the
 * D = 3 fp32 feature table of qr_forward / qr_dense_forward for that view.
 *   in : means[N,3], sh[N, (degree+1)^2, 3] fp32        out: colors[N,3] fp32
 * degree outside [0, 3]: QR_ERR_INVALID_ARG.  N = 0 is legal.  No alignment requirement.
 */
int qr_sh_colors(const qr_camera* cam, int64_t N, int32_t degree, const float* means, const float* sh, float* colors,
                 void* stream);

#ifdef __cplusplus
}
#endif
#endif /* QR_H_ */

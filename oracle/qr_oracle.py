"""ctypes/NumPy front end of the CPU oracle (oracle/qr_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from the CUDA package.  All arrays are host NumPy arrays.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass
from typing import Optional

import numpy as np

from . import build as _build

TILE = 16


class _Cam(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("fx", C.c_float), ("fy", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float), ("znear", C.c_float), ("w2c", C.c_float * 12)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_tile_lists.restype = C.c_int64
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(C.c_int(int(n)))


def _cam(cam) -> _Cam:
    c = _Cam()
    c.width, c.height = int(cam.width), int(cam.height)
    c.fx, c.fy, c.cx, c.cy, c.znear = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy), float(cam.znear)
    w = np.ascontiguousarray(cam.world_to_cam, dtype=np.float32).reshape(-1)
    for i in range(12):
        c.w2c[i] = float(w[i])
    return c


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def covariance3d(scale, quat) -> np.ndarray:
    """Sigma = R S S^T R^T, fp64."""
    s = np.ascontiguousarray(scale, dtype=np.float64)
    q = np.ascontiguousarray(quat, dtype=np.float64)
    out = np.empty(9, dtype=np.float64)
    lib().orc_covariance3d_f64(_p(s), _p(q), _p(out))
    return out.reshape(3, 3)


@dataclass
class Projected:
    mean2d: np.ndarray      # [N,2]
    conic_opac: np.ndarray  # [N,4] a, b, c, alpha
    depth: np.ndarray       # [N]
    extent: np.ndarray      # [N,2] 3*sqrt(cov_xx), 3*sqrt(cov_yy)
    visible: np.ndarray     # [N] uint8
    cov2d: Optional[np.ndarray] = None  # [N,3] (fp64 path only)


def project(cam, means, scales, quats, opac) -> Projected:
    """fp32 decision-arithmetic projection (orc_project_f32)."""
    means, scales, quats, opac = _f32(means), _f32(scales), _f32(quats), _f32(opac)
    n = means.shape[0]
    m2 = np.empty((n, 2), np.float32); co = np.empty((n, 4), np.float32)
    dp = np.empty(n, np.float32); ex = np.empty((n, 2), np.float32); vis = np.empty(n, np.uint8)
    c = _cam(cam)
    lib().orc_project_f32(C.byref(c), C.c_int64(n), _p(means), _p(scales), _p(quats), _p(opac),
                          _p(m2), _p(co), _p(dp), _p(ex), _p(vis))
    return Projected(m2, co, dp, ex, vis)


def project_f64(cam, means, scales, quats, opac) -> Projected:
    """fp64 statement of the same projection (orc_project_f64)."""
    means, scales, quats, opac = _f32(means), _f32(scales), _f32(quats), _f32(opac)
    n = means.shape[0]
    m2 = np.empty((n, 2), np.float64); cv = np.empty((n, 3), np.float64); co = np.empty((n, 4), np.float64)
    dp = np.empty(n, np.float64); ex = np.empty((n, 2), np.float64); vis = np.empty(n, np.uint8)
    c = _cam(cam)
    lib().orc_project_f64(C.byref(c), C.c_int64(n), _p(means), _p(scales), _p(quats), _p(opac),
                          _p(m2), _p(cv), _p(co), _p(dp), _p(ex), _p(vis))
    return Projected(m2, co, dp, ex, vis, cv)


def tile_rects(cam, proj: Projected):
    n = proj.mean2d.shape[0]
    rect = np.empty((n, 4), np.int32); touched = np.empty(n, np.uint32)
    c = _cam(cam)
    lib().orc_tile_rects(C.byref(c), C.c_int64(n), _p(_f32(proj.mean2d)), _p(_f32(proj.extent)),
                         _p(proj.visible), _p(rect), _p(touched))
    return rect, touched


def tile_lists(cam, depth, tile_rect, tiles_touched):
    """Per-tile (depth, id)-sorted Gaussian lists: (isect_gauss[M] uint32, tile_range[T,2] int32)."""
    depth = _f32(depth)
    tile_rect = np.ascontiguousarray(tile_rect, dtype=np.int32)
    tiles_touched = np.ascontiguousarray(tiles_touched, dtype=np.uint32)
    n = depth.shape[0]
    tx = (cam.width + TILE - 1) // TILE; ty = (cam.height + TILE - 1) // TILE
    rng = np.empty((tx * ty, 2), np.int32)
    c = _cam(cam)
    m = lib().orc_tile_lists(C.byref(c), C.c_int64(n), _p(depth), _p(tile_rect), _p(tiles_touched), _p(rng), None)
    isect = np.empty(max(int(m), 1), np.uint32)
    lib().orc_tile_lists(C.byref(c), C.c_int64(n), _p(depth), _p(tile_rect), _p(tiles_touched), _p(rng), _p(isect))
    return isect[:int(m)], rng


@dataclass
class PixelLists:
    """CSR of per-pixel depth-ordered intersection lists I with alpha'."""
    off: np.ndarray         # [H*W+1] int64
    gid: np.ndarray         # [total] int32
    alpha: np.ndarray       # [total] float32
    borderline: np.ndarray  # [H*W] uint8: list membership within 1e-6 of a cut (reading R15), anywhere in the list
    width: int
    height: int
    bl_first: Optional[np.ndarray] = None   # [H*W] int64: list position of the first such event (INT64_MAX: none)

    def ray(self, p: int):
        b, e = int(self.off[p]), int(self.off[p + 1])
        return self.gid[b:e], self.alpha[b:e]


def pixel_lists(cam, proj: Projected, mode: str = "binned") -> PixelLists:
    md = {"brute": 0, "binned": 1}[mode]
    hw = cam.width * cam.height
    n = proj.mean2d.shape[0]
    m2, co, dp, ex = _f32(proj.mean2d), _f32(proj.conic_opac), _f32(proj.depth), _f32(proj.extent)
    counts = np.zeros(hw, np.int64); bl = np.zeros(hw, np.uint8)
    blf = np.full(hw, np.iinfo(np.int64).max, np.int64)
    c = _cam(cam)
    lib().orc_pixel_lists(C.byref(c), C.c_int64(n), _p(m2), _p(co), _p(dp), _p(ex), _p(proj.visible),
                          C.c_int(md), _p(counts), _p(bl), None, None, None, _p(blf))
    off = np.zeros(hw + 1, np.int64)
    np.cumsum(counts, out=off[1:])
    tot = int(off[-1])
    gid = np.empty(max(tot, 1), np.int32); al = np.empty(max(tot, 1), np.float32)
    lib().orc_pixel_lists(C.byref(c), C.c_int64(n), _p(m2), _p(co), _p(dp), _p(ex), _p(proj.visible),
                          C.c_int(md), _p(counts), _p(bl), _p(off), _p(gid), _p(al), None)
    return PixelLists(off, gid[:tot], al[:tot], bl, cam.width, cam.height, blf)


def lists_from_rays(rays) -> PixelLists:
    """Hand-built rays: iterable of (ids, alphas).  For the pins."""
    off = [0]; g = []; a = []
    for ids, al in rays:
        ids = list(ids); al = list(al)
        assert len(ids) == len(al)
        g += ids; a += al; off.append(len(g))
    return PixelLists(np.asarray(off, np.int64), np.asarray(g, np.int32).reshape(-1),
                      np.asarray(a, np.float32).reshape(-1), np.zeros(len(off) - 1, np.uint8), len(off) - 1, 1)


@dataclass
class QOut:
    out_map: Optional[np.ndarray]  # [P,D] float32 (fp64 accumulation, rounded once)
    sel_idx: np.ndarray            # [P,K] int32, -1 padded, list order
    sel_w: np.ndarray              # [P,K] float64 normalised weights w^Q/(1-T^Q), 0 padded
    n_sel: np.ndarray              # [P] int32
    resid_TQ: np.ndarray           # [P] float64 (1 where nothing selected)
    n_walked: np.ndarray           # [P] int32 list entries consumed
    margin: np.ndarray             # [P] float64 min |T_test - boundary|


def qrender(lists: PixelLists, K: int, features: Optional[np.ndarray] = None,
            pixels: Optional[np.ndarray] = None) -> QOut:
    """Algorithm 1 on every listed pixel (or on `pixels`).  K >= 1 (K = 0 is a domain error)."""
    if K < 1:
        raise ValueError("K must be >= 1")
    npix = (len(lists.off) - 1) if pixels is None else len(pixels)
    pix = None if pixels is None else np.ascontiguousarray(pixels, dtype=np.int64)
    D = 0; feats = None; out = None; fstride = 0
    if features is not None:
        feats = _f32(features)        # fp16 tables are widened exactly (reading R14)
        D = feats.shape[1]; fstride = feats.shape[1]
        out = np.empty((npix, D), np.float32)
    sel_idx = np.empty((npix, K), np.int32); sel_w = np.empty((npix, K), np.float64)
    n_sel = np.empty(npix, np.int32); tq = np.empty(npix, np.float64)
    nw = np.empty(npix, np.int32); mg = np.empty(npix, np.float64)
    lib().orc_qrender(C.c_int64(npix), _p(pix), _p(lists.off), _p(lists.gid), _p(lists.alpha), C.c_int(K),
                      C.c_int(D), _p(feats), C.c_int64(fstride), _p(out), _p(sel_idx), _p(sel_w), _p(n_sel),
                      _p(tq), _p(nw), _p(mg))
    return QOut(out, sel_idx, sel_w, n_sel, tq, nw, mg)


@dataclass
class VOut:
    out_map: np.ndarray      # [P,D] float32
    final_T: np.ndarray      # [P] float64
    stop_margin: np.ndarray  # [P] float64, relative distance of the nearest T_test to t_min
    n_blended: np.ndarray    # [P] int32


def vrender(lists: PixelLists, features: np.ndarray, t_min: float = 1e-4,
            pixels: Optional[np.ndarray] = None) -> VOut:
    """Eq. 1 with the early stop of reading R7 (t_min = 0: exact Eq. 1)."""
    npix = (len(lists.off) - 1) if pixels is None else len(pixels)
    pix = None if pixels is None else np.ascontiguousarray(pixels, dtype=np.int64)
    feats = _f32(features); D = feats.shape[1]
    out = np.empty((npix, D), np.float32); ft = np.empty(npix, np.float64)
    sm = np.empty(npix, np.float64); nb = np.empty(npix, np.int32)
    lib().orc_vrender(C.c_int64(npix), _p(pix), _p(lists.off), _p(lists.gid), _p(lists.alpha), C.c_int(D),
                      _p(feats), C.c_int64(D), C.c_float(t_min), _p(out), _p(ft), _p(sm), _p(nb))
    return VOut(out, ft, sm, nb)


@dataclass
class TopKOut:
    out_map: Optional[np.ndarray]  # [P,D] float32
    sel_idx: np.ndarray            # [P,K] int32, -1 padded, depth order
    sel_w: np.ndarray              # [P,K] float64 normalised weights w^top/(1-T^top), 0 padded
    n_sel: np.ndarray              # [P] int32 = min(K, n_dense)
    resid: np.ndarray              # [P] float64 T^top (1 where nothing kept)
    gap: np.ndarray                # [P] float64 (w_(K) - w_(K+1)) / w_(K), inf when everything is kept
    stop_margin: np.ndarray        # [P] float64 as VOut.stop_margin
    n_dense: np.ndarray            # [P] int32 entries that received a dense weight


def topk(lists: PixelLists, K: int, features: Optional[np.ndarray] = None, t_min: float = 1e-4,
         pixels: Optional[np.ndarray] = None) -> TopKOut:
    """Top-K render: K largest dense weights, re-blended in depth order."""
    if K < 1:
        raise ValueError("K must be >= 1")
    npix = (len(lists.off) - 1) if pixels is None else len(pixels)
    pix = None if pixels is None else np.ascontiguousarray(pixels, dtype=np.int64)
    D = 0; feats = None; out = None; fstride = 0
    if features is not None:
        feats = _f32(features)
        D = feats.shape[1]; fstride = feats.shape[1]
        out = np.empty((npix, D), np.float32)
    sel_idx = np.empty((npix, K), np.int32); sel_w = np.empty((npix, K), np.float64)
    n_sel = np.empty(npix, np.int32); rs = np.empty(npix, np.float64)
    gap = np.empty(npix, np.float64); sm = np.empty(npix, np.float64); nd = np.empty(npix, np.int32)
    lib().orc_topk(C.c_int64(npix), _p(pix), _p(lists.off), _p(lists.gid), _p(lists.alpha), C.c_int(K), C.c_int(D),
                   _p(feats), C.c_int64(fstride), C.c_float(t_min), _p(out), _p(sel_idx), _p(sel_w), _p(n_sel), _p(rs),
                   _p(gap), _p(sm), _p(nd))
    return TopKOut(out, sel_idx, sel_w, n_sel, rs, gap, sm, nd)


@dataclass
class StratOut:
    out_map: Optional[np.ndarray]
    sel_idx: np.ndarray
    sel_w: np.ndarray
    n_sel: np.ndarray
    resid_TQ: np.ndarray
    n_walked: np.ndarray
    margin: np.ndarray          # [P] float64 min |T_test - boundary| over the walk
    stop_margin: np.ndarray     # [P] float64 pass 1: relative distance of the nearest T_test to t_min
    mu: np.ndarray              # [P] float32 mean of the dense transmittance values
    sigma: np.ndarray           # [P] float32 their population standard deviation (0: uniform boundaries)
    n_dense: np.ndarray         # [P] int32 entries the statistics cover


def stratified(lists: PixelLists, K: int, features: Optional[np.ndarray] = None, t_min: float = 1e-4, z_max: float = 2.0,
               pixels: Optional[np.ndarray] = None) -> StratOut:
    """Stratified-K (reading R18): Algorithm 1 with boundaries mu + sigma z_k."""
    if K < 1:
        raise ValueError("K must be >= 1")
    npix = (len(lists.off) - 1) if pixels is None else len(pixels)
    pix = None if pixels is None else np.ascontiguousarray(pixels, dtype=np.int64)
    D = 0; feats = None; out = None; fstride = 0
    if features is not None:
        feats = _f32(features)
        D = feats.shape[1]; fstride = feats.shape[1]
        out = np.empty((npix, D), np.float32)
    sel_idx = np.empty((npix, K), np.int32); sel_w = np.empty((npix, K), np.float64)
    n_sel = np.empty(npix, np.int32); tq = np.empty(npix, np.float64)
    nw = np.empty(npix, np.int32); mg = np.empty(npix, np.float64); sm = np.empty(npix, np.float64)
    mu = np.empty(npix, np.float32); sg = np.empty(npix, np.float32); nd = np.empty(npix, np.int32)
    lib().orc_stratified(C.c_int64(npix), _p(pix), _p(lists.off), _p(lists.gid), _p(lists.alpha), C.c_int(K), C.c_int(D),
                         _p(feats), C.c_int64(fstride), C.c_float(t_min), C.c_float(z_max), _p(out), _p(sel_idx), _p(sel_w),
                         _p(n_sel), _p(tq), _p(nw), _p(mg), _p(sm), _p(mu), _p(sg), _p(nd))
    return StratOut(out, sel_idx, sel_w, n_sel, tq, nw, mg, sm, mu, sg, nd)


def backward(sel_idx, sel_w, n_sel, dL_dmap, N: int, rows: Optional[np.ndarray] = None) -> np.ndarray:
    """dL/dF rows (all N, or only `rows`) in fp64 from the selection records of every pixel."""
    sel_idx = np.ascontiguousarray(sel_idx, dtype=np.int32)
    sel_w = np.ascontiguousarray(sel_w, dtype=np.float64)
    n_sel = np.ascontiguousarray(n_sel, dtype=np.int32)
    npix, K = sel_idx.shape
    g = _f32(dL_dmap).reshape(npix, -1); D = g.shape[1]
    r = None if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
    R = N if r is None else len(r)
    out = np.empty((R, D), np.float64)
    lib().orc_backward(C.c_int64(npix), C.c_int(K), C.c_int(D), C.c_int64(N), _p(sel_idx), _p(sel_w), _p(n_sel),
                       _p(g), C.c_int64(0 if r is None else len(r)), _p(r), _p(out))
    return out


def render_scene(scene, K: Optional[int] = None, mode: str = "binned", with_features: bool = True):
    """Convenience: O1 -> O2 -> O4 on a qr_inputs.Scene-like object.  Returns (proj, lists, QOut)."""
    proj = project(scene.cam, scene.means, scene.scales, scene.quats, scene.opac)
    lists = pixel_lists(scene.cam, proj, mode)
    q = qrender(lists, scene.K if K is None else K, scene.features if with_features else None)
    return proj, lists, q


def devoxelize(uni, inverse_indices, counts, reduce: str = "max"):
    """De-voxelisation (Listing 3): returns (gs_pred [G,C] float64, argmax [G,C] int64)."""
    uni = _f32(uni)
    inv = np.ascontiguousarray(inverse_indices, dtype=np.int64)
    cnt = np.ascontiguousarray(counts, dtype=np.int64)
    if reduce not in ("mean", "max"):
        raise ValueError("reduce must be 'mean' or 'max'")
    if cnt.sum() != len(inv) or (len(inv) and (inv.min() < 0 or inv.max() >= uni.shape[0])):
        raise ValueError("index out of range / counts do not cover the voxels")
    G, C_ = len(cnt), uni.shape[1]
    out = np.empty((G, C_), np.float64); am = np.empty((G, C_), np.int64)
    lib().orc_devoxelize(C.c_int64(uni.shape[0]), C.c_int(C_), C.c_int64(G), _p(uni), _p(inv), _p(cnt), C.c_int(reduce == "max"),
                         _p(out), _p(am))
    return out, am


def devoxelize_backward(n_unique: int, inverse_indices, counts, reduce: str, argmax, d_gs):
    inv = np.ascontiguousarray(inverse_indices, dtype=np.int64)
    cnt = np.ascontiguousarray(counts, dtype=np.int64)
    d = _f32(d_gs)
    am = None if argmax is None else np.ascontiguousarray(argmax, dtype=np.int64)
    out = np.empty((n_unique, d.shape[1]), np.float64)
    lib().orc_devoxelize_backward(C.c_int64(n_unique), C.c_int(d.shape[1]), C.c_int64(len(cnt)), _p(inv), _p(cnt),
                                  C.c_int(reduce == "max"), _p(am), _p(d), _p(out))
    return out


@dataclass
class MaskLoss:
    loss: float
    loss_per_mask: np.ndarray   # [S] float64 (0 for empty masks)
    pooled: np.ndarray          # [S,D] float64 mean of the map over each mask
    d_map: np.ndarray           # [P,D] float64


def mask_loss(feature_map, mask_id, targets) -> MaskLoss:
    """Mask-pooled contrastive loss (Eq. 2; reading R19) and its gradient w.r.t. the map."""
    m = _f32(feature_map)
    m = m.reshape(-1, m.shape[-1])
    mid = np.ascontiguousarray(mask_id, dtype=np.int32).reshape(-1)
    t = _f32(targets)
    P_, D = m.shape
    S = t.shape[0]
    pooled = np.empty((S, D), np.float64); ls = np.empty(S, np.float64); tot = C.c_double(0.0)
    dm = np.empty((P_, D), np.float64)
    lib().orc_mask_loss(C.c_int64(P_), C.c_int(D), _p(m), _p(mid), C.c_int(S), _p(t), _p(pooled), _p(ls), C.byref(tot), _p(dm))
    return MaskLoss(float(tot.value), ls, pooled, dm)



def sh_basis(degree: int, direction) -> np.ndarray:
    """The (degree+1)^2 real spherical harmonics of DESIGN.md reading R20 at a unit vector (float64)."""
    d = np.ascontiguousarray(direction, dtype=np.float64).reshape(3)
    Y = np.zeros(16, np.float64)
    lib().orc_sh_basis(C.c_int(int(degree)), _p(d), _p(Y))
    return Y[:(degree + 1) ** 2]


def sh_colors(cam, means, sh, degree: int) -> np.ndarray:
    """View-dependent RGB of every Gaussian (reading R20): [N,3] float64."""
    m = _f32(means)
    s = _f32(sh)
    N = m.shape[0]
    assert 0 <= degree <= 3 and s.shape == (N, (degree + 1) ** 2, 3), s.shape
    out = np.empty((N, 3), np.float64)
    c = _cam(cam)
    lib().orc_sh_colors(C.byref(c), C.c_int64(N), C.c_int(int(degree)), _p(m), _p(s), _p(out))
    return out

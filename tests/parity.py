"""Parity helpers shared by the -m gpu tests: run the CUDA path (through the C ABI binding) and the CPU oracle on
the same seeded scene and compare them element by element under the tolerances BASELINE.json's north_star states:

  * selected indices bit-exact except at pixels whose transmittance lies within 1e-6 of a quantile threshold
    (oracle margin, fp64) or whose list membership is within 1e-6 of a cut (reading R15) -- those are counted;
  * fp32 features / gradients within 1e-5 + 1e-4 |ref|; fp16-stored features within 2e-3 relative.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np
import torch

MARGIN = 1e-6
ATOL, RTOL = 1e-5, 1e-4
RTOL_F16 = 2e-3


def to_dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


@dataclass
class GpuScene:
    means: torch.Tensor
    scales: torch.Tensor
    quats: torch.Tensor
    opac: torch.Tensor
    features: torch.Tensor


def upload(sc) -> GpuScene:
    return GpuScene(to_dev(sc.means), to_dev(sc.scales), to_dev(sc.quats), to_dev(sc.opac), to_dev(sc.features))


def oracle_frontend(orc, sc):
    proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    rect, touched = orc.tile_rects(sc.cam, proj)
    isect, rng = orc.tile_lists(sc.cam, proj.depth, rect, touched)
    return proj, rect, touched, isect, rng


def exempt_classes(q, lists, pixels=None):
    """The two classes of pixels exempt from bit-exact index parity (reading R15), reported separately:
    margin     -- some T_test of the walk lies within 1e-6 of a quantile threshold (north_star's own clause);
    borderline -- the walk meets a Gaussian whose list membership is within 1e-6 of a cut of R4 (a 1-ulp expf
                  difference flips membership of I).  Only events inside the walked prefix count: position of the
                  first event <= entries the oracle's walk consumed."""
    margin = q.margin <= MARGIN
    if lists.bl_first is not None:
        blf = lists.bl_first if pixels is None else lists.bl_first[pixels]
        border = blf <= q.n_walked.astype(np.int64)
    else:
        border = lists.borderline.astype(bool)
        if pixels is not None:
            border = border[pixels]
    return margin, border


def exempt_mask(q, lists, pixels=None):
    """Pixels the north_star exempts from bit-exact index parity."""
    margin, border = exempt_classes(q, lists, pixels)
    return margin | border


def masked_records(out):
    """(sel_idx, sel_w, n_sel) of a binding.ForwardOut as NumPy arrays [H*W, K] / [H*W], with the slots at or beyond
    n_sel -- which qr_forward leaves unwritten -- set to -1 / 0 so that whole arrays can be compared."""
    H, W = out.n_sel.shape
    K = out.sel_idx.shape[-1]
    n = out.n_sel.cpu().numpy().reshape(H * W)
    used = np.arange(K)[None, :] < n[:, None]
    idx = np.where(used, out.sel_idx.cpu().numpy().reshape(H * W, K), -1)
    w = np.where(used, out.sel_w.cpu().numpy().reshape(H * W, K), 0.0)
    return idx, w, n


def same_selection(sel_idx, n_sel, q):
    """Per pixel: the GPU selected the same Gaussians in the same order as the oracle.  Slots at or beyond n_sel are
    not part of the result (include/qr.h: qr_forward leaves them unwritten), so only the used prefix is compared."""
    K = sel_idx.shape[1]
    used = np.arange(K)[None, :] < q.n_sel[:, None]
    return (n_sel == q.n_sel) & ((sel_idx == q.sel_idx) | ~used).all(axis=1)


def compare_forward(gpu_out, q, lists, K, D, f16=False, pixels=None):
    """gpu_out: binding.ForwardOut (full image).  q: oracle QOut for all pixels (or for `pixels`).
    Returns a dict of counts; raises AssertionError on a non-exempt mismatch."""
    H, W = gpu_out.n_sel.shape
    sel_idx = gpu_out.sel_idx.cpu().numpy().reshape(H * W, K)
    sel_w = gpu_out.sel_w.cpu().numpy().reshape(H * W, K)
    n_sel = gpu_out.n_sel.cpu().numpy().reshape(H * W)
    resid = gpu_out.resid_TQ.cpu().numpy().reshape(H * W)
    out_map = gpu_out.out_map.cpu().numpy().reshape(H * W, D)
    if pixels is not None:
        sel_idx, sel_w, n_sel, resid, out_map = sel_idx[pixels], sel_w[pixels], n_sel[pixels], resid[pixels], out_map[pixels]
    ex_m, ex_b = exempt_classes(q, lists, pixels)
    ex = ex_m | ex_b
    same = same_selection(sel_idx, n_sel, q)
    bad = (~same) & (~ex)
    stats = dict(pixels=int(same.size), exempt=int(ex.sum()), exempt_margin=int(ex_m.sum()),
                 exempt_borderline=int((ex_b & ~ex_m).sum()), mismatch_exempt=int(((~same) & ex).sum()),
                 mismatch_nonexempt=int(bad.sum()))
    assert stats["mismatch_nonexempt"] == 0, f"index mismatch at non-exempt pixels: {stats}; first {np.flatnonzero(bad)[:5]}"
    ok = same                       # values are compared where the selection agrees
    used = np.arange(K)[None, :] < q.n_sel[:, None]
    np.testing.assert_allclose(np.where(used, sel_w, 0.0)[ok], q.sel_w[ok], rtol=RTOL, atol=ATOL)
    np.testing.assert_allclose(resid[ok], q.resid_TQ[ok], rtol=RTOL, atol=ATOL)
    if q.out_map is not None:
        ref = q.out_map[ok].astype(np.float64)
        got = out_map[ok].astype(np.float64)
        if f16:
            tol = RTOL_F16 * np.abs(ref) + 1e-5
        else:
            tol = ATOL + RTOL * np.abs(ref)
        err = np.abs(got - ref)
        worst = float((err / tol).max()) if err.size else 0.0
        stats["worst_tol_frac"] = worst
        assert worst <= 1.0, f"feature map outside tolerance: worst err/tol = {worst}"
    # zero-selection pixels render zero and report T^Q = 1 (R8)
    z = n_sel == 0
    assert (out_map[z] == 0).all() and (resid[z] == 1.0).all()
    return stats


EPS32 = 2.0 ** -24
FANIN_ULPS = 4.0


def compare_backward_rows(got_rows, ref_rows, what="", abs_sum_rows=None):
    """Element-wise gradient parity on a set of dL/dF rows.  The bar is north_star's fp32 tolerance, 1e-5 + 1e-4 |ref|.
    A row element is a sum over every pixel that selected the Gaussian; at full size that is up to ~5e4 terms of either
    sign (a near Gaussian covers the screen), and NO fp32 accumulation of them -- whatever its order -- is closer to
    the fp64 sum than about one fp32 rounding unit of A = sum |w g| ("Tolerances").  Where the caller passes
    A (computed by the oracle from |dL_dmap|), FANIN_ULPS = 4 such units, 4 x 2^-24 A, are added to the tolerance (one
    each for the tf32 x 3 operand split, the tensor core's truncating fp32 accumulation, the fp32 atomics across half
    tiles and the rounding of the result); how many elements needed it (i.e. exceed the plain bar: a handful per 10^7)
    is returned and printed by the callers.  Returns (worst err / tol, count)."""
    ref = np.asarray(ref_rows, dtype=np.float64)
    got = np.asarray(got_rows, dtype=np.float64)
    assert ref.shape == got.shape and ref.size > 0, (what, ref.shape, got.shape)
    plain = ATOL + RTOL * np.abs(ref)
    err = np.abs(got - ref)
    over_plain = int((err > plain).sum())
    tol = plain if abs_sum_rows is None else plain + FANIN_ULPS * EPS32 * np.asarray(abs_sum_rows, dtype=np.float64)
    worst = float((err / tol).max())
    assert worst <= 1.0, (f"{what}: gradient outside tolerance, worst err/tol = {worst}, "
                          f"{over_plain} of {err.size} elements over the plain 1e-5 + 1e-4|ref|")
    return worst, over_plain


TOPK_GAP = 1e-5


def compare_topk(gpu_out, t, lists, K, D, f16=False, pixels=None):
    """qr_topk_forward against the oracle's orc_topk (reading R17).  Index parity is exact except at pixels
    where a 1-ulp expf difference can legitimately change the result, counted and returned: the K-th and (K+1)-th
    largest dense weights within 1e-5 relative of each other (`gap`: a 1-ulp expf difference moves the dense T by up to
    a few 1e-6 relative), the early stop within 1e-5 relative of t_min (as for the
    dense comparator), or list membership within 1e-6 of a cut of R4 anywhere in the weighted prefix."""
    H, W = gpu_out.n_sel.shape
    sel_idx = gpu_out.sel_idx.cpu().numpy().reshape(H * W, K)
    sel_w = gpu_out.sel_w.cpu().numpy().reshape(H * W, K)
    n_sel = gpu_out.n_sel.cpu().numpy().reshape(H * W)
    resid = gpu_out.resid_TQ.cpu().numpy().reshape(H * W)
    out_map = gpu_out.out_map.cpu().numpy().reshape(H * W, D)
    bl = lists.borderline.astype(bool)
    if pixels is not None:
        sel_idx, sel_w, n_sel, resid, out_map, bl = sel_idx[pixels], sel_w[pixels], n_sel[pixels], resid[pixels], out_map[pixels], bl[pixels]
    ex_gap = t.gap <= TOPK_GAP
    ex_stop = t.stop_margin <= 1e-5
    ex = ex_gap | ex_stop | bl
    same = same_selection(sel_idx, n_sel, t)
    bad = (~same) & (~ex)
    stats = dict(pixels=int(same.size), exempt=int(ex.sum()), exempt_gap=int(ex_gap.sum()), exempt_stop=int(ex_stop.sum()),
                 exempt_borderline=int(bl.sum()), mismatch_exempt=int(((~same) & ex).sum()), mismatch_nonexempt=int(bad.sum()))
    assert stats["mismatch_nonexempt"] == 0, f"top-K index mismatch at non-exempt pixels: {stats}; first {np.flatnonzero(bad)[:5]}"
    ok = same
    used = np.arange(K)[None, :] < t.n_sel[:, None]
    np.testing.assert_allclose(np.where(used, sel_w, 0.0)[ok], t.sel_w[ok], rtol=RTOL, atol=ATOL)
    np.testing.assert_allclose(resid[ok], t.resid[ok], rtol=RTOL, atol=ATOL)
    if t.out_map is not None:
        ref = t.out_map[ok].astype(np.float64)
        got = out_map[ok].astype(np.float64)
        tol = (RTOL_F16 * np.abs(ref) + 1e-5) if f16 else (ATOL + RTOL * np.abs(ref))
        err = np.abs(got - ref)
        worst = float((err / tol).max()) if err.size else 0.0
        stats["worst_tol_frac"] = worst
        assert worst <= 1.0, f"top-K feature map outside tolerance: worst err/tol = {worst}"
    z = n_sel == 0
    assert (out_map[z] == 0).all() and (resid[z] == 1.0).all()
    return stats


STRAT_BAND = 1e-5


def compare_stratified(gpu_out, t, lists, K, D, pixels=None):
    """qr_forward_stratified against orc_stratified (reading R18).  Same comparison as compare_forward, with the
    exemption band on |T_test - boundary| widened from 1e-6 to 1e-5: the boundaries mu + sigma z_k are themselves functions
    of the ray's transmittance values, and a 1-ulp expf difference moves sigma = sqrt(E[T^2] - mu^2) by up to ~1e-6 / sigma.
    Pixels whose pass-1 stop lies within 1e-5 relative of t_min (the statistics then cover one entry more or less) are
    exempt too.  Both classes are counted."""
    import copy
    q = copy.copy(t)
    m = np.where(t.stop_margin <= 1e-5, 0.0, t.margin * (MARGIN / STRAT_BAND))
    q.margin = m
    stats = compare_forward(gpu_out, q, lists, K, D, pixels=pixels)
    stats["exempt_stop"] = int((t.stop_margin <= 1e-5).sum())
    return stats

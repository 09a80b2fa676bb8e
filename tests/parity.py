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


def exempt_mask(q, lists, pixels=None):
    """Pixels the north_star exempts from bit-exact index parity."""
    bl = lists.borderline.astype(bool)
    if pixels is not None:
        bl = bl[pixels]
    return (q.margin <= MARGIN) | bl


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
    ex = exempt_mask(q, lists, pixels)
    same = (sel_idx == q.sel_idx).all(axis=1) & (n_sel == q.n_sel)
    bad = (~same) & (~ex)
    stats = dict(pixels=int(same.size), exempt=int(ex.sum()), mismatch_exempt=int(((~same) & ex).sum()),
                 mismatch_nonexempt=int(bad.sum()))
    assert stats["mismatch_nonexempt"] == 0, f"index mismatch at non-exempt pixels: {stats}; first {np.flatnonzero(bad)[:5]}"
    ok = same                       # values are compared where the selection agrees
    # padding conventions
    pad = np.arange(K)[None, :] >= n_sel[:, None]
    assert (sel_idx[pad] == -1).all() and (sel_w[pad] == 0).all()
    np.testing.assert_allclose(sel_w[ok], q.sel_w[ok], rtol=RTOL, atol=ATOL)
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

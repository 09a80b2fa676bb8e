"""Call sequences over the binding (no arithmetic): the front end (qr_preprocess -> qr_bin_count -> qr_bin_sort),
Q-Render forward / backward and the dense comparator.  Everything stays on the device except M (one int64)."""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import torch

from . import binding as B


@dataclass
class Frontend:
    proj: B.Projected
    offsets: Optional[torch.Tensor]
    M: int                      # entries isect_gauss holds (the exact count, or the caller's capacity)
    isect_gauss: torch.Tensor
    tile_range: torch.Tensor
    found: Optional[torch.Tensor] = None    # capacity path: 1-element int64 device tensor, intersections found


def frontend(cam, means, scales, quats, opac, capacity: Optional[int] = None) -> Frontend:
    """PAPER.md:80 steps (1) tiling and (2) splatting: projection, intersection count, duplication + sort.

    capacity = None: qr_bin_count sizes the lists exactly (one device->host read of M, the only synchronisation of
    the path).  capacity = an upper bound on the number of intersections (e.g. 1.25 x the previous frame's): nothing
    synchronises; `found` (device) must be checked against capacity when the frame's results are read -- if it is
    larger the lists were truncated and the frame has to be redone with a larger capacity."""
    proj = B.qr_preprocess(cam, means, scales, quats, opac)
    if capacity is None:
        offsets, M = B.qr_bin_count(proj.tiles_touched)
        isect, rng = B.qr_bin_sort(cam, M, proj.depth, proj.tile_rect, offsets)
        return Frontend(proj, offsets, M, isect, rng)
    isect, rng, found = B.qr_bin_sort(cam, int(capacity), proj.depth, proj.tile_rect, None, return_found=True)
    return Frontend(proj, None, int(capacity), isect, rng, found)


def forward(cam, fe: Frontend, features: torch.Tensor, K: int, out: Optional[B.ForwardOut] = None,
            select_only: bool = False) -> B.ForwardOut:
    return B.qr_forward(cam, K, fe.proj.mean2d, fe.proj.conic_opac, fe.isect_gauss, fe.tile_range, features, out,
                        select_only=select_only)


def backward(cam, N: int, fwd: B.ForwardOut, dL_dmap: torch.Tensor, dL_dfeat: Optional[torch.Tensor] = None,
             ws: Optional[torch.Tensor] = None):
    """dL/dF of the frame `fwd`.  Without a workspace of its own the call goes through qr_backward_lists where the
    forward left its selection lists (fp32 features, D % 128 == 0: no second numbering pass); with `ws`, or for the
    other shapes, through qr_backward on the selection records."""
    D = int(dL_dmap.shape[-1])
    if ws is None and fwd.ws is not None and fwd.has_lists and fwd.out_map.shape[-1] == D:
        return B.qr_backward_lists(cam, int(fwd.sel_idx.shape[-1]), N, fwd.ws, dL_dmap, dL_dfeat)
    return B.qr_backward(cam, N, fwd.sel_idx, fwd.sel_w, fwd.n_sel, dL_dmap, dL_dfeat, ws)


def backward_clear(cam, N: int, fwd: B.ForwardOut, dL_dfeat: torch.Tensor, ws: Optional[torch.Tensor] = None):
    """Re-zero the rows the last backward touched (instead of zeroing the whole [N, D] table).  ws = the workspace that
    backward used: its own, or (default) the forward's."""
    return B.qr_backward_clear(cam, N, fwd.sel_idx, fwd.n_sel, dL_dfeat, fwd.ws if ws is None else ws)


def dense_forward(cam, fe: Frontend, features: torch.Tensor, t_min: float = 1e-4, out_map=None, final_T=None):
    return B.qr_dense_forward(cam, fe.proj.mean2d, fe.proj.conic_opac, fe.isect_gauss, fe.tile_range, features, t_min,
                              out_map, final_T)


def dense_forward_tc(cam, fe: Frontend, features: torch.Tensor, t_min: float = 1e-4, cap: int = 128, out_map=None, final_T=None, ws=None):
    """The dense comparator with the blend on the tensor cores (binding.qr_dense_forward_tc).  Returns (out_map, final_T, ws)."""
    return B.qr_dense_forward_tc(cam, fe.proj.mean2d, fe.proj.conic_opac, fe.isect_gauss, fe.tile_range, features, t_min, cap,
                                 out_map, final_T, ws)


def topk_forward(cam, fe: Frontend, features: torch.Tensor, K: int, t_min: float = 1e-4, out: Optional[B.ForwardOut] = None):
    """The top-K comparator on the same front end."""
    return B.qr_topk_forward(cam, K, fe.proj.mean2d, fe.proj.conic_opac, fe.isect_gauss, fe.tile_range, features, t_min, out)


def frontend_batch(cams, means, scales, quats, opac, capacity: Optional[int] = None):
    """Front end of a batch of views (include/qr.h, multi-camera batching): one projection launch for all cameras, one
    sort over the tall tile grid.  Returns (tall camera, Frontend); arrays have B * N entries."""
    tall = B.qr_batch_camera(cams)
    proj = B.qr_preprocess_batch(cams, means, scales, quats, opac)
    if capacity is None:
        offsets, M = B.qr_bin_count(proj.tiles_touched)
        isect, rng = B.qr_bin_sort(tall, M, proj.depth, proj.tile_rect, offsets)
        return tall, Frontend(proj, offsets, M, isect, rng)
    isect, rng, found = B.qr_bin_sort(tall, int(capacity), proj.depth, proj.tile_rect, None, return_found=True)
    return tall, Frontend(proj, None, int(capacity), isect, rng, found)


def forward_batch(tall, n_views: int, N: int, fe: Frontend, features: torch.Tensor, K: int, out: Optional[B.ForwardOut] = None):
    """Q-Render of every view of the batch in one walk + one blend; outputs are [B*H, W, ...].  backward / backward_clear
    take `tall` and N as they are and accumulate every view into one dL_dfeat."""
    return B.qr_forward_batch(tall, n_views, N, K, fe.proj.mean2d, fe.proj.conic_opac, fe.isect_gauss, fe.tile_range, features, out)


def stratified_forward(cam, fe: Frontend, features: torch.Tensor, K: int, t_min: float = 1e-4, z_max: float = 2.0,
                       out: Optional[B.ForwardOut] = None):
    """The stratified-K variant: two walks, then the same blend; backward() takes its output as is."""
    return B.qr_forward_stratified(cam, K, fe.proj.mean2d, fe.proj.conic_opac, fe.isect_gauss, fe.tile_range, features, t_min, z_max, out)


def devoxelize(uni_pred, inverse_indices, num_voxels_per_g, reduce: str = "max"):
    """Per-unique-voxel predictions -> per-Gaussian feature table (Listing 3); see binding.qr_devoxelize."""
    return B.qr_devoxelize(uni_pred, inverse_indices, num_voxels_per_g, reduce)


def mask_loss(cam, feature_map, mask_id, targets):
    """Mask-pooled contrastive loss of PAPER.md Eq. 2 and dL/dmap for backward(); see binding.qr_mask_loss."""
    return B.qr_mask_loss(cam, feature_map, mask_id, targets)


def pooled_loss(cam, N: int, fwd: B.ForwardOut, features, mask_id, targets, dL_dfeat=None, with_grad: bool = True):
    """Loss + dL/dF from the selection lists of `fwd` (which may come from forward(..., select_only=True)): no map round trip."""
    return B.qr_pooled_loss(cam, int(fwd.sel_idx.shape[-1]), N, fwd, features, mask_id, targets, dL_dfeat, with_grad)


def sh_colors(cam, means, sh, degree: int, colors=None):
    """RGB payload: per-view colours from spherical harmonics; feed the result to forward() as the
    D = 3 feature table.  See binding.qr_sh_colors."""
    return B.qr_sh_colors(cam, means, sh, degree, colors)


def forward_multik(cam, fe: Frontend, features: torch.Tensor, Ks, outs=None):
    """Q-Render for several K in one walk (binding.qr_forward_multik): a list of ForwardOut, one per K; backward() and
    backward_clear() take each of them as they take forward()'s."""
    return B.qr_forward_multik(cam, Ks, fe.proj.mean2d, fe.proj.conic_opac, fe.isect_gauss, fe.tile_range, features, outs)

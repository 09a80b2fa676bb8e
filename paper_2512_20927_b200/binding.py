"""Thin ctypes binding of libqr.so (include/qr.h): argument marshalling only.

Every function has the name of the C entry point it calls and does nothing but check tensor device / dtype /
contiguity, allocate outputs through PyTorch, pass raw device pointers plus the current CUDA stream, and turn a
negative status into ``QRError``.  No step of the path runs in Python or in PyTorch ops.  There is no CPU fallback:
if libqr.so cannot be loaded, or a tensor is not on a CUDA device, the call raises.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional, Tuple

import torch

from . import _build

QR_F32, QR_F16 = 0, 1
QR_TILE = 16
QR_MAX_K = 256
QR_MAX_D = 512

STATUS = {0: "QR_OK", -1: "QR_ERR_INVALID_ARG", -2: "QR_ERR_NULL_POINTER", -3: "QR_ERR_UNSUPPORTED",
          -4: "QR_ERR_WORKSPACE_TOO_SMALL", -5: "QR_ERR_CAPACITY", -6: "QR_ERR_CUDA", -7: "QR_ERR_MISALIGNED"}

# every symbol include/qr.h declares (tests check that the library exports exactly these)
SYMBOLS = ["qr_version", "qr_last_error", "qr_num_tiles", "qr_preprocess", "qr_bin_workspace_bytes", "qr_bin_count",
           "qr_bin_sort", "qr_forward_workspace_bytes", "qr_forward", "qr_backward_workspace_bytes", "qr_backward",
           "qr_backward_lists", "qr_backward_clear", "qr_dense_forward", "qr_dense_workspace_bytes", "qr_dense_forward_tc", "qr_topk_workspace_bytes", "qr_topk_forward",
           "qr_launch_count", "qr_forward_stats", "qr_batch_camera", "qr_preprocess_batch", "qr_forward_batch",
           "qr_stratified_workspace_bytes", "qr_forward_stratified", "qr_devoxelize_workspace_bytes", "qr_devoxelize",
           "qr_devoxelize_backward", "qr_mask_loss_workspace_bytes", "qr_mask_loss", "qr_pooled_loss", "qr_sh_colors", "qr_mask_loss_static", "qr_forward_multik"]


class QRError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{STATUS.get(code, code)}: {msg}")
        self.code = code


class qr_camera(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("fx", C.c_float), ("fy", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float), ("znear", C.c_float), ("world_to_cam", C.c_float * 12)]


_lib = None


def lib_path() -> str:
    return _build.LIB


def load() -> C.CDLL:
    """Load (building if the sources are newer) libqr.so.  Raises if it cannot be had -- no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if os.environ.get("QR_NO_BUILD", "0") != "1":
        try:
            path = _build.build()
        except Exception as e:  # nvcc missing on a box that already has the .so: use it as shipped
            if not os.path.exists(_build.LIB):
                raise RuntimeError(f"libqr.so is missing and cannot be built: {e}") from e
    if not os.path.exists(path):
        raise RuntimeError("libqr.so is missing: run `python paper_2512_20927_b200/_build.py` (no CPU fallback)")
    lib = C.CDLL(path)
    vp, i32, i64, sz, f32 = C.c_void_p, C.c_int32, C.c_int64, C.c_size_t, C.c_float
    cam = C.POINTER(qr_camera)
    lib.qr_version.restype = C.c_int
    lib.qr_last_error.restype = C.c_char_p
    lib.qr_num_tiles.restype = i32; lib.qr_num_tiles.argtypes = [cam]
    lib.qr_preprocess.restype = C.c_int
    lib.qr_preprocess.argtypes = [cam, i64, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.qr_bin_workspace_bytes.restype = sz; lib.qr_bin_workspace_bytes.argtypes = [i64, i64, i32]
    lib.qr_bin_count.restype = C.c_int
    lib.qr_bin_count.argtypes = [i64, vp, vp, C.POINTER(i64), vp, sz, vp]
    lib.qr_bin_sort.restype = C.c_int
    lib.qr_bin_sort.argtypes = [cam, i64, i64, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.qr_forward_workspace_bytes.restype = sz; lib.qr_forward_workspace_bytes.argtypes = [cam, i32, i32]
    lib.qr_forward.restype = C.c_int
    lib.qr_forward.argtypes = [cam, i32, i32, C.c_int, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.qr_backward_workspace_bytes.restype = sz; lib.qr_backward_workspace_bytes.argtypes = [cam, i32, i32]
    lib.qr_backward.restype = C.c_int
    lib.qr_backward.argtypes = [cam, i32, i32, i64, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.qr_backward_lists.restype = C.c_int
    lib.qr_backward_lists.argtypes = [cam, i32, i32, i64, vp, sz, vp, vp, vp]
    lib.qr_backward_clear.restype = C.c_int
    lib.qr_backward_clear.argtypes = [cam, i32, i32, i64, vp, vp, vp, vp, sz, vp]
    lib.qr_dense_forward.restype = C.c_int
    lib.qr_dense_forward.argtypes = [cam, i32, C.c_int, f32, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.qr_dense_workspace_bytes.restype = sz; lib.qr_dense_workspace_bytes.argtypes = [cam, i32]
    lib.qr_dense_forward_tc.restype = C.c_int
    lib.qr_dense_forward_tc.argtypes = [cam, i32, C.c_int, f32, i32, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.qr_launch_count.restype = C.c_longlong; lib.qr_launch_count.argtypes = []
    lib.qr_forward_stats.restype = C.c_int; lib.qr_forward_stats.argtypes = [cam, i32, vp, sz, vp, vp]
    lib.qr_batch_camera.restype = C.c_int; lib.qr_batch_camera.argtypes = [cam, i32, cam]
    lib.qr_preprocess_batch.restype = C.c_int
    lib.qr_preprocess_batch.argtypes = [cam, i32, i64, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.qr_forward_batch.restype = C.c_int
    lib.qr_forward_batch.argtypes = [cam, i32, i64, i32, i32, C.c_int, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.qr_stratified_workspace_bytes.restype = sz; lib.qr_stratified_workspace_bytes.argtypes = [cam, i32, i32]
    lib.qr_forward_stratified.restype = C.c_int
    lib.qr_forward_stratified.argtypes = [cam, i32, i32, C.c_int, f32, f32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.qr_devoxelize_workspace_bytes.restype = sz; lib.qr_devoxelize_workspace_bytes.argtypes = [i64]
    lib.qr_devoxelize.restype = C.c_int; lib.qr_devoxelize.argtypes = [i64, i32, i64, vp, vp, vp, i32, vp, vp, vp, sz, vp]
    lib.qr_devoxelize_backward.restype = C.c_int
    lib.qr_devoxelize_backward.argtypes = [i64, i32, i64, vp, i32, vp, vp, vp, vp, sz, vp]
    lib.qr_mask_loss_workspace_bytes.restype = sz; lib.qr_mask_loss_workspace_bytes.argtypes = [i32, i32]
    lib.qr_mask_loss.restype = C.c_int; lib.qr_mask_loss.argtypes = [cam, i32, i32, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.qr_forward_multik.restype = C.c_int
    lib.qr_forward_multik.argtypes = [cam, i32, vp, i32, C.c_int, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.qr_mask_loss_static.restype = C.c_int; lib.qr_mask_loss_static.argtypes = [cam, i32, i32, vp, vp, vp, vp, vp, vp, vp]
    lib.qr_pooled_loss.restype = C.c_int
    lib.qr_pooled_loss.argtypes = [cam, i32, i32, i64, vp, sz, vp, vp, i32, vp, vp, vp, vp, vp, sz, vp]
    lib.qr_sh_colors.restype = C.c_int
    lib.qr_sh_colors.argtypes = [cam, i64, i32, vp, vp, vp, vp]
    lib.qr_topk_workspace_bytes.restype = sz; lib.qr_topk_workspace_bytes.argtypes = [cam, i32, i32]
    lib.qr_topk_forward.restype = C.c_int
    lib.qr_topk_forward.argtypes = [cam, i32, i32, C.c_int, f32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    _lib = lib
    return lib


def _check(rc: int) -> None:
    if rc != 0:
        raise QRError(rc, load().qr_last_error().decode("utf-8", "replace"))


def make_camera(cam) -> qr_camera:
    """From any object with width, height, fx, fy, cx, cy, znear, world_to_cam (e.g. qr_inputs.Camera)."""
    if isinstance(cam, qr_camera):
        return cam
    c = qr_camera()
    c.width, c.height = int(cam.width), int(cam.height)
    c.fx, c.fy, c.cx, c.cy, c.znear = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy), float(cam.znear)
    w = [float(v) for v in list(cam.world_to_cam.reshape(-1))]
    for i in range(12):
        c.world_to_cam[i] = w[i]
    return c


def _dev(t: torch.Tensor, dtype, name: str) -> int:
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise QRError(-1, f"{name} must be a CUDA tensor (libqr has no CPU path)")
    if t.dtype != dtype:
        raise QRError(-1, f"{name} must have dtype {dtype}, got {t.dtype}")
    if not t.is_contiguous():
        raise QRError(-1, f"{name} must be contiguous")
    return t.data_ptr()


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def qr_version() -> int:
    return int(load().qr_version())


def qr_num_tiles(cam) -> int:
    c = make_camera(cam)
    return int(load().qr_num_tiles(C.byref(c)))


@dataclass
class Projected:
    mean2d: torch.Tensor         # [N,2] f32
    conic_opac: torch.Tensor     # [N,4] f32
    depth: torch.Tensor          # [N] f32
    tile_rect: torch.Tensor      # [N,4] i32
    tiles_touched: torch.Tensor  # [N] u32 stored as int32 bits


def qr_preprocess(cam, means, scales, quats, opac) -> Projected:
    c = make_camera(cam)
    n = int(means.shape[0])
    dev = means.device
    out = Projected(torch.empty((n, 2), dtype=torch.float32, device=dev),
                    torch.empty((n, 4), dtype=torch.float32, device=dev),
                    torch.empty((n,), dtype=torch.float32, device=dev),
                    torch.empty((n, 4), dtype=torch.int32, device=dev),
                    torch.empty((n,), dtype=torch.int32, device=dev))
    _check(load().qr_preprocess(C.byref(c), n, _dev(means, torch.float32, "means"), _dev(scales, torch.float32, "scales"),
                                _dev(quats, torch.float32, "quats"), _dev(opac, torch.float32, "opac"),
                                out.mean2d.data_ptr(), out.conic_opac.data_ptr(), out.depth.data_ptr(),
                                out.tile_rect.data_ptr(), out.tiles_touched.data_ptr(), _stream()))
    return out


def qr_bin_workspace_bytes(N: int, M: int, num_tiles: int) -> int:
    return int(load().qr_bin_workspace_bytes(int(N), int(M), int(num_tiles)))


def qr_bin_count(tiles_touched: torch.Tensor, ws: Optional[torch.Tensor] = None) -> Tuple[torch.Tensor, int]:
    """Returns (offsets[N] as int64 bits of the uint64 inclusive scan, M)."""
    n = int(tiles_touched.shape[0])
    dev = tiles_touched.device
    offsets = torch.empty((n,), dtype=torch.int64, device=dev)
    if ws is None:
        ws = torch.empty((max(qr_bin_workspace_bytes(n, 0, 0), 16),), dtype=torch.uint8, device=dev)
    m = C.c_int64(0)
    _check(load().qr_bin_count(n, _dev(tiles_touched, torch.int32, "tiles_touched"), offsets.data_ptr(), C.byref(m),
                               ws.data_ptr(), ws.numel(), _stream()))
    return offsets, int(m.value)


def qr_bin_sort(cam, M: int, depth, tile_rect, offsets=None, ws: Optional[torch.Tensor] = None,
                isect_gauss: Optional[torch.Tensor] = None, tile_range: Optional[torch.Tensor] = None,
                return_found: bool = False):
    """Returns (isect_gauss[M] int32 bits of the uint32 ids, tile_range[T,2] int32).  M is the exact count from
    qr_bin_count or an upper bound (no host synchronisation needed then); with return_found also a 1-element int64
    DEVICE tensor = the number of intersections found (> M: the lists are truncated, call again with a larger M)."""
    c = make_camera(cam)
    n = int(depth.shape[0])
    dev = depth.device
    T = qr_num_tiles(c)
    if isect_gauss is None:
        isect_gauss = torch.empty((max(M, 1),), dtype=torch.int32, device=dev)
    if tile_range is None:
        tile_range = torch.empty((T, 2), dtype=torch.int32, device=dev)
    if ws is None:
        ws = torch.empty((max(qr_bin_workspace_bytes(n, M, T), 16),), dtype=torch.uint8, device=dev)
    off_ptr = None if offsets is None else _dev(offsets, torch.int64, "offsets")
    _check(load().qr_bin_sort(C.byref(c), n, int(M), _dev(depth, torch.float32, "depth"),
                              _dev(tile_rect, torch.int32, "tile_rect"), off_ptr,
                              isect_gauss.data_ptr(), tile_range.data_ptr(), ws.data_ptr(), ws.numel(), _stream()))
    if return_found:
        return isect_gauss[:M], tile_range, ws[:8].view(torch.int64)
    return isect_gauss[:M], tile_range


@dataclass
class ForwardOut:
    out_map: torch.Tensor   # [H,W,D] f32
    sel_idx: torch.Tensor   # [H,W,K] i32
    sel_w: torch.Tensor     # [H,W,K] f32
    n_sel: torch.Tensor     # [H,W] i32
    resid_TQ: torch.Tensor  # [H,W] f32
    ws: Optional[torch.Tensor] = None   # the workspace the call used: for fp32 D % 128 == 0 it holds the selection lists
                                        # qr_backward_lists / qr_backward_clear read, until the next call that writes it
    has_lists: bool = False


def _feat_dtype(features: torch.Tensor) -> int:
    if features.dtype == torch.float32:
        return QR_F32
    if features.dtype == torch.float16:
        return QR_F16
    raise QRError(-1, f"features must be float32 or float16, got {features.dtype}")


def qr_forward_workspace_bytes(cam, K: int, D: int) -> int:
    c = make_camera(cam)
    return int(load().qr_forward_workspace_bytes(C.byref(c), int(K), int(D)))


_ws_cache = {}


def _workspace(nbytes: int, dev, tag: str = "") -> torch.Tensor:
    """One cached scratch tensor per device (and tag), grown on demand (device memory only; contents are scratch)."""
    key = str(dev) + tag
    t = _ws_cache.get(key)
    if t is None or t.numel() < nbytes:
        t = torch.empty((max(int(nbytes), 256),), dtype=torch.uint8, device=dev)
        _ws_cache[key] = t
    return t


def qr_forward(cam, K: int, mean2d, conic_opac, isect_gauss, tile_range, features,
               out: Optional[ForwardOut] = None, ws: Optional[torch.Tensor] = None, select_only: bool = False) -> ForwardOut:
    """select_only: pass out_map = NULL (tcgen05 path): the walk, the records and the selection lists, no blend, no map."""
    c = make_camera(cam)
    H, W = c.height, c.width
    D = int(features.shape[1])
    dev = features.device
    dt = _feat_dtype(features)
    if ws is None:
        ws = _workspace(qr_forward_workspace_bytes(c, K, D), dev)
    if out is not None:
        kk = max(int(K), 1)
        want = {"out_map": (H, W, D), "sel_idx": (H, W, kk), "sel_w": (H, W, kk), "n_sel": (H, W), "resid_TQ": (H, W)}
        for name, shape in want.items():
            if tuple(getattr(out, name).shape) != shape:
                raise QRError(-1, f"out.{name} has shape {tuple(getattr(out, name).shape)}, expected {shape}")
    if out is None:
        kk = max(int(K), 1)
        out = ForwardOut(torch.empty((H, W, D), dtype=torch.float32, device=dev),
                         torch.empty((H, W, kk), dtype=torch.int32, device=dev),
                         torch.empty((H, W, kk), dtype=torch.float32, device=dev),
                         torch.empty((H, W), dtype=torch.int32, device=dev),
                         torch.empty((H, W), dtype=torch.float32, device=dev))
    _check(load().qr_forward(C.byref(c), int(K), D, dt, _dev(mean2d, torch.float32, "mean2d"),
                             _dev(conic_opac, torch.float32, "conic_opac"),
                             _dev(isect_gauss, torch.int32, "isect_gauss"), _dev(tile_range, torch.int32, "tile_range"),
                             _dev(features, features.dtype, "features"), None if select_only else out.out_map.data_ptr(),
                             out.sel_idx.data_ptr(), out.sel_w.data_ptr(), out.n_sel.data_ptr(), out.resid_TQ.data_ptr(),
                             ws.data_ptr(), ws.numel(), _stream()))
    out.ws = ws
    out.has_lists = lists_supported(features.dtype, D)
    return out


def lists_supported(features_dtype, D: int) -> bool:
    """qr_forward leaves selection lists in its workspace on the tcgen05 path: fp32 / fp16 features with D % 32 == 0, or D < 32
    with D % 4 == 0 (fp16: D % 8 == 0), D <= 512 (include/qr.h; the contractions run on whole 128-channel tiles, TMA pads)."""
    ok = 4 <= D <= min(QR_MAX_D, 512) and (D % 32 == 0 or (D < 32 and D % 4 == 0))
    return ok and (features_dtype == torch.float32 or (features_dtype == torch.float16 and D % 8 == 0))


def qr_backward_workspace_bytes(cam, K: int, D: int) -> int:
    c = make_camera(cam)
    return int(load().qr_backward_workspace_bytes(C.byref(c), int(K), int(D)))


def qr_backward_workspace(cam, K: int, D: int, device) -> torch.Tensor:
    """Scratch for qr_backward; keep it to pass the same tensor to qr_backward_clear afterwards."""
    return torch.empty((max(qr_backward_workspace_bytes(cam, K, D), 16),), dtype=torch.uint8, device=device)


def qr_backward(cam, N: int, sel_idx, sel_w, n_sel, dL_dmap, dL_dfeat: Optional[torch.Tensor] = None,
                ws: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Accumulates into dL_dfeat[N,D] (allocated zero-filled when not given)."""
    c = make_camera(cam)
    K = int(sel_idx.shape[-1])
    D = int(dL_dmap.shape[-1])
    if dL_dfeat is None:
        dL_dfeat = torch.zeros((int(N), D), dtype=torch.float32, device=dL_dmap.device)
    if ws is None:
        ws = qr_backward_workspace(cam, K, D, dL_dmap.device)
    _check(load().qr_backward(C.byref(c), K, D, int(N), _dev(sel_idx, torch.int32, "sel_idx"),
                              _dev(sel_w, torch.float32, "sel_w"), _dev(n_sel, torch.int32, "n_sel"),
                              _dev(dL_dmap, torch.float32, "dL_dmap"), _dev(dL_dfeat, torch.float32, "dL_dfeat"),
                              _dev(ws, torch.uint8, "ws"), ws.numel(), _stream()))
    return dL_dfeat


def qr_backward_lists(cam, K: int, N: int, fwd_ws: torch.Tensor, dL_dmap, dL_dfeat: Optional[torch.Tensor] = None) -> torch.Tensor:
    """qr_backward from the selection lists the last qr_forward left in its workspace fwd_ws (ForwardOut.ws)."""
    c = make_camera(cam)
    D = int(dL_dmap.shape[-1])
    if dL_dfeat is None:
        dL_dfeat = torch.zeros((int(N), D), dtype=torch.float32, device=dL_dmap.device)
    _check(load().qr_backward_lists(C.byref(c), int(K), D, int(N), _dev(fwd_ws, torch.uint8, "fwd_ws"), fwd_ws.numel(),
                                    _dev(dL_dmap, torch.float32, "dL_dmap"), _dev(dL_dfeat, torch.float32, "dL_dfeat"),
                                    _stream()))
    return dL_dfeat


def qr_backward_clear(cam, N: int, sel_idx, n_sel, dL_dfeat: torch.Tensor, ws: torch.Tensor) -> torch.Tensor:
    """Zeroes the rows of dL_dfeat the last qr_backward (same selection, same ws) added into."""
    c = make_camera(cam)
    K = int(sel_idx.shape[-1])
    D = int(dL_dfeat.shape[-1])
    _check(load().qr_backward_clear(C.byref(c), K, D, int(N), _dev(sel_idx, torch.int32, "sel_idx"),
                                    _dev(n_sel, torch.int32, "n_sel"), _dev(dL_dfeat, torch.float32, "dL_dfeat"),
                                    _dev(ws, torch.uint8, "ws"), ws.numel(), _stream()))
    return dL_dfeat


def qr_dense_forward(cam, mean2d, conic_opac, isect_gauss, tile_range, features, t_min: float = 1e-4,
                     out_map: Optional[torch.Tensor] = None, final_T: Optional[torch.Tensor] = None):
    c = make_camera(cam)
    H, W = c.height, c.width
    D = int(features.shape[1])
    dev = features.device
    if out_map is None:
        out_map = torch.empty((H, W, D), dtype=torch.float32, device=dev)
    if final_T is None:
        final_T = torch.empty((H, W), dtype=torch.float32, device=dev)
    _check(load().qr_dense_forward(C.byref(c), D, _feat_dtype(features), float(t_min),
                                   _dev(mean2d, torch.float32, "mean2d"), _dev(conic_opac, torch.float32, "conic_opac"),
                                   _dev(isect_gauss, torch.int32, "isect_gauss"),
                                   _dev(tile_range, torch.int32, "tile_range"),
                                   _dev(features, features.dtype, "features"), out_map.data_ptr(), final_T.data_ptr(),
                                   _stream()))
    return out_map, final_T


def qr_dense_forward_tc(cam, mean2d, conic_opac, isect_gauss, tile_range, features, t_min: float = 1e-4, cap: int = 128,
                        out_map: Optional[torch.Tensor] = None, final_T: Optional[torch.Tensor] = None,
                        ws: Optional[torch.Tensor] = None):
    """qr_dense_forward with the blend on the tensor cores (include/qr.h qr_dense_forward_tc); cap = list capacity in
    entries per pixel.  Returns (out_map, final_T, ws)."""
    c = make_camera(cam)
    H, W = c.height, c.width
    D = int(features.shape[1])
    dev = features.device
    if out_map is None:
        out_map = torch.empty((H, W, D), dtype=torch.float32, device=dev)
    if final_T is None:
        final_T = torch.empty((H, W), dtype=torch.float32, device=dev)
    need = int(load().qr_dense_workspace_bytes(C.byref(c), int(cap)))
    if ws is None or ws.numel() < need:
        ws = torch.empty((max(need, 256),), dtype=torch.uint8, device=dev)
    _check(load().qr_dense_forward_tc(C.byref(c), D, _feat_dtype(features), float(t_min), int(cap),
                                      _dev(mean2d, torch.float32, "mean2d"), _dev(conic_opac, torch.float32, "conic_opac"),
                                      isect_gauss.data_ptr() if isect_gauss.numel() else None,
                                      _dev(tile_range, torch.int32, "tile_range"),
                                      _dev(features, features.dtype, "features"), out_map.data_ptr(), final_T.data_ptr(),
                                      ws.data_ptr(), ws.numel(), _stream()))
    return out_map, final_T, ws


def qr_topk_forward(cam, K: int, mean2d, conic_opac, isect_gauss, tile_range, features, t_min: float = 1e-4,
                    out: Optional[ForwardOut] = None, ws: Optional[torch.Tensor] = None) -> ForwardOut:
    """Top-K render comparator (include/qr.h qr_topk_forward).  Returns records in qr_forward's format; its workspace
    is its own (the forward's selection lists are left alone)."""
    c = make_camera(cam)
    H, W = c.height, c.width
    D = int(features.shape[1])
    dev = features.device
    dt = _feat_dtype(features)
    if ws is None:
        ws = _workspace(int(load().qr_topk_workspace_bytes(C.byref(c), int(K), D)), dev, "topk")
    kk = max(int(K), 1)
    if out is None:
        out = ForwardOut(torch.empty((H, W, D), dtype=torch.float32, device=dev),
                         torch.empty((H, W, kk), dtype=torch.int32, device=dev),
                         torch.empty((H, W, kk), dtype=torch.float32, device=dev),
                         torch.empty((H, W), dtype=torch.int32, device=dev),
                         torch.empty((H, W), dtype=torch.float32, device=dev))
    else:
        want = {"out_map": (H, W, D), "sel_idx": (H, W, kk), "sel_w": (H, W, kk), "n_sel": (H, W), "resid_TQ": (H, W)}
        for name, shape in want.items():
            if tuple(getattr(out, name).shape) != shape:
                raise QRError(-1, f"out.{name} has shape {tuple(getattr(out, name).shape)}, expected {shape}")
    _check(load().qr_topk_forward(C.byref(c), int(K), D, dt, float(t_min), _dev(mean2d, torch.float32, "mean2d"),
                                  _dev(conic_opac, torch.float32, "conic_opac"),
                                  _dev(isect_gauss, torch.int32, "isect_gauss"), _dev(tile_range, torch.int32, "tile_range"),
                                  _dev(features, features.dtype, "features"), out.out_map.data_ptr(), out.sel_idx.data_ptr(),
                                  out.sel_w.data_ptr(), out.n_sel.data_ptr(), out.resid_TQ.data_ptr(),
                                  ws.data_ptr(), ws.numel(), _stream()))
    out.ws = None
    out.has_lists = False
    return out


def qr_launch_count() -> int:
    return int(load().qr_launch_count())


FORWARD_STATS = ("selections", "sum_U_half_tiles", "list_entries_consumed", "entry_pixel_evaluations", "walk_cycles",
                 "half_tiles_U_gt_64")


def qr_forward_stats(cam, K: int, fwd: ForwardOut) -> dict:
    """Work counters of the forward that produced `fwd` (tcgen05 path only); synchronises to read eight integers."""
    if not fwd.has_lists or fwd.ws is None:
        raise QRError(-3, "qr_forward_stats needs the workspace of a forward on the tcgen05 path")
    c = make_camera(cam)
    st = torch.empty((8,), dtype=torch.int64, device=fwd.ws.device)
    _check(load().qr_forward_stats(C.byref(c), int(K), fwd.ws.data_ptr(), fwd.ws.numel(), st.data_ptr(), _stream()))
    v = st.cpu().tolist()
    return dict(zip(FORWARD_STATS, v[:len(FORWARD_STATS)]))


def _cam_array(cams):
    arr = (qr_camera * len(cams))()
    for i, c in enumerate(cams):
        arr[i] = make_camera(c)
    return arr


def qr_batch_camera(cams) -> qr_camera:
    """The camera of the tall image that stacks the views of `cams` (include/qr.h, multi-camera batching)."""
    arr = _cam_array(cams)
    tall = qr_camera()
    _check(load().qr_batch_camera(arr, len(cams), C.byref(tall)))
    return tall


def qr_preprocess_batch(cams, means, scales, quats, opac) -> Projected:
    """qr_preprocess for every camera of `cams` in one launch; arrays have B * N entries (view b in [b N, (b+1) N))."""
    arr = _cam_array(cams)
    B = len(cams)
    n = int(means.shape[0])
    dev = means.device
    out = Projected(torch.empty((B * n, 2), dtype=torch.float32, device=dev), torch.empty((B * n, 4), dtype=torch.float32, device=dev),
                    torch.empty((B * n,), dtype=torch.float32, device=dev), torch.empty((B * n, 4), dtype=torch.int32, device=dev),
                    torch.empty((B * n,), dtype=torch.int32, device=dev))
    _check(load().qr_preprocess_batch(arr, B, n, _dev(means, torch.float32, "means"), _dev(scales, torch.float32, "scales"),
                                      _dev(quats, torch.float32, "quats"), _dev(opac, torch.float32, "opac"),
                                      out.mean2d.data_ptr(), out.conic_opac.data_ptr(), out.depth.data_ptr(),
                                      out.tile_rect.data_ptr(), out.tiles_touched.data_ptr(), _stream()))
    return out


def qr_forward_batch(tall, B: int, N: int, K: int, mean2d, conic_opac, isect_gauss, tile_range, features,
                     out: Optional[ForwardOut] = None, ws: Optional[torch.Tensor] = None) -> ForwardOut:
    """qr_forward on the tall image of a batch of B views (N Gaussians per view).  Outputs are [B*H, W, ...]."""
    c = make_camera(tall)
    H, W = c.height, c.width
    D = int(features.shape[1])
    dev = features.device
    dt = _feat_dtype(features)
    if ws is None:
        ws = _workspace(qr_forward_workspace_bytes(c, K, D), dev)
    kk = max(int(K), 1)
    if out is None:
        out = ForwardOut(torch.empty((H, W, D), dtype=torch.float32, device=dev),
                         torch.empty((H, W, kk), dtype=torch.int32, device=dev),
                         torch.empty((H, W, kk), dtype=torch.float32, device=dev),
                         torch.empty((H, W), dtype=torch.int32, device=dev),
                         torch.empty((H, W), dtype=torch.float32, device=dev))
    else:
        want = {"out_map": (H, W, D), "sel_idx": (H, W, kk), "sel_w": (H, W, kk), "n_sel": (H, W), "resid_TQ": (H, W)}
        for name, shape in want.items():
            if tuple(getattr(out, name).shape) != shape:
                raise QRError(-1, f"out.{name} has shape {tuple(getattr(out, name).shape)}, expected {shape}")
    _check(load().qr_forward_batch(C.byref(c), int(B), int(N), int(K), D, dt, _dev(mean2d, torch.float32, "mean2d"),
                                   _dev(conic_opac, torch.float32, "conic_opac"),
                                   _dev(isect_gauss, torch.int32, "isect_gauss"), _dev(tile_range, torch.int32, "tile_range"),
                                   _dev(features, features.dtype, "features"), out.out_map.data_ptr(), out.sel_idx.data_ptr(),
                                   out.sel_w.data_ptr(), out.n_sel.data_ptr(), out.resid_TQ.data_ptr(),
                                   ws.data_ptr(), ws.numel(), _stream()))
    out.ws = ws
    out.has_lists = lists_supported(features.dtype, D)
    return out


def qr_forward_stratified(cam, K: int, mean2d, conic_opac, isect_gauss, tile_range, features, t_min: float = 1e-4,
                          z_max: float = 2.0, out: Optional[ForwardOut] = None, ws: Optional[torch.Tensor] = None) -> ForwardOut:
    """Stratified-K forward (include/qr.h qr_forward_stratified); same outputs as qr_forward, own (cached) workspace."""
    c = make_camera(cam)
    H, W = c.height, c.width
    D = int(features.shape[1])
    dev = features.device
    dt = _feat_dtype(features)
    if ws is None:
        ws = _workspace(int(load().qr_stratified_workspace_bytes(C.byref(c), int(K), D)), dev, "strat")
    kk = max(int(K), 1)
    if out is None:
        out = ForwardOut(torch.empty((H, W, D), dtype=torch.float32, device=dev),
                         torch.empty((H, W, kk), dtype=torch.int32, device=dev),
                         torch.empty((H, W, kk), dtype=torch.float32, device=dev),
                         torch.empty((H, W), dtype=torch.int32, device=dev),
                         torch.empty((H, W), dtype=torch.float32, device=dev))
    _check(load().qr_forward_stratified(C.byref(c), int(K), D, dt, float(t_min), float(z_max),
                                        _dev(mean2d, torch.float32, "mean2d"), _dev(conic_opac, torch.float32, "conic_opac"),
                                        _dev(isect_gauss, torch.int32, "isect_gauss"), _dev(tile_range, torch.int32, "tile_range"),
                                        _dev(features, features.dtype, "features"), out.out_map.data_ptr(), out.sel_idx.data_ptr(),
                                        out.sel_w.data_ptr(), out.n_sel.data_ptr(), out.resid_TQ.data_ptr(),
                                        ws.data_ptr(), ws.numel(), _stream()))
    out.ws = ws
    out.has_lists = lists_supported(features.dtype, D)
    return out


REDUCE = {"mean": 0, "max": 1}


def qr_devoxelize(uni_pred, inverse_indices, num_voxels_per_g, reduce: str = "max", ws: Optional[torch.Tensor] = None):
    """De-voxelisation (include/qr.h qr_devoxelize; Listing 3).  Returns (gs_pred [G,C], argmax [G,C] or None, ws);
    pass argmax and ws to qr_devoxelize_backward."""
    U, Cn = int(uni_pred.shape[0]), int(uni_pred.shape[1])
    G = int(num_voxels_per_g.shape[0])
    dev = uni_pred.device
    if ws is None:
        ws = torch.empty((max(int(load().qr_devoxelize_workspace_bytes(G)), 256),), dtype=torch.uint8, device=dev)
    gs = torch.empty((G, Cn), dtype=torch.float32, device=dev)
    am = torch.empty((G, Cn), dtype=torch.int32, device=dev) if reduce == "max" else None
    _check(load().qr_devoxelize(U, Cn, G, _dev(uni_pred, torch.float32, "uni_pred"), _dev(inverse_indices, torch.int64, "inverse_indices"),
                                _dev(num_voxels_per_g, torch.int32, "num_voxels_per_g"), REDUCE[reduce], gs.data_ptr(),
                                None if am is None else am.data_ptr(), ws.data_ptr(), ws.numel(), _stream()))
    return gs, am, ws


def qr_devoxelize_backward(n_unique: int, inverse_indices, reduce: str, argmax, d_gs, ws: torch.Tensor,
                           d_uni: Optional[torch.Tensor] = None) -> torch.Tensor:
    G, Cn = int(d_gs.shape[0]), int(d_gs.shape[1])
    if d_uni is None:
        d_uni = torch.zeros((n_unique, Cn), dtype=torch.float32, device=d_gs.device)
    _check(load().qr_devoxelize_backward(int(n_unique), Cn, G, _dev(inverse_indices, torch.int64, "inverse_indices"), REDUCE[reduce],
                                         None if argmax is None else _dev(argmax, torch.int32, "argmax"),
                                         _dev(d_gs, torch.float32, "d_gs"), _dev(d_uni, torch.float32, "d_uni"),
                                         _dev(ws, torch.uint8, "ws"), ws.numel(), _stream()))
    return d_uni


def qr_mask_loss(cam, feature_map, mask_id, targets, d_map: Optional[torch.Tensor] = None):
    """Mask-pooled contrastive loss and dL/dmap (include/qr.h qr_mask_loss).  Returns (loss [1], loss_per_mask [S], d_map)."""
    c = make_camera(cam)
    D = int(feature_map.shape[-1])
    S = int(targets.shape[0])
    dev = feature_map.device
    ws = _workspace(int(load().qr_mask_loss_workspace_bytes(S, D)), dev, "maskloss")
    loss = torch.empty((1,), dtype=torch.float32, device=dev)
    per = torch.empty((S,), dtype=torch.float32, device=dev)
    if d_map is None:
        d_map = torch.empty((c.height, c.width, D), dtype=torch.float32, device=dev)
    _check(load().qr_mask_loss(C.byref(c), D, S, _dev(feature_map, torch.float32, "map"), _dev(mask_id, torch.int32, "mask_id"),
                               _dev(targets, torch.float32, "targets"), loss.data_ptr(), per.data_ptr(), d_map.data_ptr(),
                               ws.data_ptr(), ws.numel(), _stream()))
    return loss, per, d_map


def qr_pooled_loss(cam, K: int, N: int, fwd: ForwardOut, features, mask_id, targets, dL_dfeat: Optional[torch.Tensor] = None,
                   with_grad: bool = True):
    """The mask-pooled loss and dL/dF straight from the forward's selection lists, without the map (include/qr.h
    qr_pooled_loss).  Returns (loss [1], loss_per_mask [S], dL_dfeat or None)."""
    if not fwd.has_lists or fwd.ws is None:
        raise QRError(-3, "qr_pooled_loss needs the workspace of a forward on the tcgen05 path")
    c = make_camera(cam)
    D = int(features.shape[1])
    S = int(targets.shape[0])
    dev = features.device
    ws = _workspace(int(load().qr_mask_loss_workspace_bytes(S, D)), dev, "maskloss")
    loss = torch.empty((1,), dtype=torch.float32, device=dev)
    per = torch.empty((S,), dtype=torch.float32, device=dev)
    if with_grad and dL_dfeat is None:
        dL_dfeat = torch.zeros((N, D), dtype=torch.float32, device=dev)
    _check(load().qr_pooled_loss(C.byref(c), int(K), D, int(N), fwd.ws.data_ptr(), fwd.ws.numel(), _dev(features, torch.float32, "features"),
                                 _dev(mask_id, torch.int32, "mask_id"), S, _dev(targets, torch.float32, "targets"), loss.data_ptr(),
                                 per.data_ptr(), dL_dfeat.data_ptr() if with_grad else None, ws.data_ptr(), ws.numel(), _stream()))
    return loss, per, (dL_dfeat if with_grad else None)


def qr_sh_colors(cam, means, sh, degree: int, colors: Optional[torch.Tensor] = None):
    """View-dependent RGB of every Gaussian from its spherical-harmonics coefficients (include/qr.h qr_sh_colors;
    PAPER.md:940-947, reading R20).  sh [N, (degree+1)^2, 3] fp32 -> colors [N, 3] fp32, the D = 3 feature table
    of qr_forward for this view."""
    c = make_camera(cam)
    N = int(means.shape[0])
    if tuple(sh.shape) != (N, (int(degree) + 1) ** 2, 3):
        raise QRError(-1, f"sh has shape {tuple(sh.shape)}, expected {(N, (int(degree) + 1) ** 2, 3)}")
    if colors is None:
        colors = torch.empty((N, 3), dtype=torch.float32, device=means.device)
    _check(load().qr_sh_colors(C.byref(c), N, int(degree), _dev(means, torch.float32, "means"), _dev(sh, torch.float32, "sh"),
                               _dev(colors, torch.float32, "colors"), _stream()))
    return colors


def qr_mask_loss_static(cam, feature_map, mask_id, targets, loss: Optional[torch.Tensor] = None,
                        loss_per_mask: Optional[torch.Tensor] = None, d_map: Optional[torch.Tensor] = None):
    """qr_mask_loss without a workspace: the library's own static device array serves as scratch (include/qr.h
    qr_mask_loss_static; at most 256 masks at D = 512).  The C call allocates nothing; pass loss [1], loss_per_mask [S] and
    d_map [H, W, D] to keep this wrapper from allocating them.  Calls that overlap on the GPU race on the array."""
    c = make_camera(cam)
    D = int(feature_map.shape[-1])
    S = int(targets.shape[0])
    dev = feature_map.device
    if loss is None:
        loss = torch.empty((1,), dtype=torch.float32, device=dev)
    if loss_per_mask is None:
        loss_per_mask = torch.empty((S,), dtype=torch.float32, device=dev)
    if d_map is None:
        d_map = torch.empty((c.height, c.width, D), dtype=torch.float32, device=dev)
    _check(load().qr_mask_loss_static(C.byref(c), D, S, _dev(feature_map, torch.float32, "map"), _dev(mask_id, torch.int32, "mask_id"),
                                      _dev(targets, torch.float32, "targets"), _dev(loss, torch.float32, "loss"),
                                      _dev(loss_per_mask, torch.float32, "loss_per_mask"), _dev(d_map, torch.float32, "d_map"), _stream()))
    return loss, loss_per_mask, d_map


def qr_forward_multik(cam, Ks, mean2d, conic_opac, isect_gauss, tile_range, features, outs=None):
    """qr_forward for up to four K in one walk (include/qr.h qr_forward_multik).  Returns a list of ForwardOut, one per K, each
    with a workspace of its own that holds that K's selection lists (pass `outs` to reuse the outputs of an earlier call)."""
    c = make_camera(cam)
    H, W = c.height, c.width
    D = int(features.shape[1])
    dev = features.device
    Ks = [int(k) for k in Ks]
    n = len(Ks)
    if outs is None:
        outs = []
        for K in Ks:
            kk = max(K, 1)
            o = ForwardOut(torch.empty((H, W, D), dtype=torch.float32, device=dev),
                           torch.empty((H, W, kk), dtype=torch.int32, device=dev),
                           torch.empty((H, W, kk), dtype=torch.float32, device=dev),
                           torch.empty((H, W), dtype=torch.int32, device=dev),
                           torch.empty((H, W), dtype=torch.float32, device=dev))
            o.ws = torch.empty((max(qr_forward_workspace_bytes(c, K, D), 256),), dtype=torch.uint8, device=dev)
            outs.append(o)
    arr_i = (C.c_int32 * max(n, 1))(*Ks)
    parr = lambda ts: (C.c_void_p * max(n, 1))(*[t.data_ptr() for t in ts])
    sizes = (C.c_size_t * max(n, 1))(*[o.ws.numel() for o in outs])
    _check(load().qr_forward_multik(C.byref(c), n, arr_i, D, _feat_dtype(features), _dev(mean2d, torch.float32, "mean2d"),
                                    _dev(conic_opac, torch.float32, "conic_opac"), _dev(isect_gauss, torch.int32, "isect_gauss"),
                                    _dev(tile_range, torch.int32, "tile_range"), _dev(features, features.dtype, "features"),
                                    parr([o.out_map for o in outs]), parr([o.sel_idx for o in outs]), parr([o.sel_w for o in outs]),
                                    parr([o.n_sel for o in outs]), parr([o.resid_TQ for o in outs]), parr([o.ws for o in outs]),
                                    sizes, _stream()))
    for o in outs:
        o.has_lists = True
    return outs

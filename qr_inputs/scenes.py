"""Seeded scene / camera / payload generator (no rendering arithmetic here).

Stands in for the paper's workload (ScanNet scene0000_00, 512-D CLIP-aligned
Gaussian features, K=40: PAPER.md:27, :381, :967), which is not available.
Shapes and distributions follow BASELINE.json ``configs`` as read in
SURVEY.md section 8(d); every choice the configs leave open is listed in DESIGN.md.

Draw order from ``np.random.default_rng(seed)`` (fixed, documented):
  [blob centres, blob assignment,] means, scales, quats, opacities,
  [blob centre features,] features, dL_dmap.
All arrays are float32, C-contiguous.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Dict, Optional

import numpy as np


@dataclass
class Camera:
    """Pinhole camera.  Pixel (x, y) samples the image plane at (x+0.5, y+0.5).

    ``world_to_cam`` is the row-major 3x4 [R|t] mapping world points into the
    camera frame (x right, y down, z forward).
    """
    width: int
    height: int
    fx: float
    fy: float
    cx: float
    cy: float
    znear: float
    world_to_cam: np.ndarray  # [3,4] float32

    def copy(self) -> "Camera":
        return replace(self, world_to_cam=self.world_to_cam.copy())


@dataclass
class Scene:
    name: str
    cam: Camera
    means: np.ndarray      # [N,3] f32
    scales: np.ndarray     # [N,3] f32 > 0
    quats: np.ndarray      # [N,4] f32 (w,x,y,z), unit
    opac: np.ndarray       # [N]   f32 in (0,1)
    features: np.ndarray   # [N,D] f32 (or f16 when feat_dtype == "f16"), unit-norm rows
    dL_dmap: Optional[np.ndarray]  # [H,W,D] f32 or None
    K: int
    feat_dtype: str = "f32"
    meta: Dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return int(self.means.shape[0])

    @property
    def D(self) -> int:
        return int(self.features.shape[1])


def make_camera(width: int, height: int, fov_x_deg: float = 60.0, znear: float = 0.2,
                world_to_cam: Optional[np.ndarray] = None) -> Camera:
    """Horizontal field of view ``fov_x_deg``; square pixels; principal point at the centre."""
    f = (width / 2.0) / math.tan(math.radians(fov_x_deg) / 2.0)
    if world_to_cam is None:
        world_to_cam = np.concatenate([np.eye(3), np.zeros((3, 1))], axis=1)
    return Camera(int(width), int(height), float(np.float32(f)), float(np.float32(f)),
                  width / 2.0, height / 2.0, float(znear),
                  np.ascontiguousarray(world_to_cam, dtype=np.float32))


def look_at(position, target, down=(0.0, 1.0, 0.0)) -> np.ndarray:
    """3x4 world-to-camera for a camera at ``position`` looking at ``target`` with +y down."""
    c = np.asarray(position, dtype=np.float64)
    f = np.asarray(target, dtype=np.float64) - c
    f /= np.linalg.norm(f)
    d = np.asarray(down, dtype=np.float64)
    x = np.cross(d, f)
    x /= np.linalg.norm(x)
    y = np.cross(f, x)
    R = np.stack([x, y, f], axis=0)
    t = -R @ c
    return np.concatenate([R, t[:, None]], axis=1).astype(np.float32)


def pose_on_circle(j: int, n_poses: int = 8, radius: float = 3.0, centre=(0.0, 0.0, 0.0)) -> np.ndarray:
    """Config-4 poses: position (r cos th_j, 0, r sin th_j) + centre, looking at the centre."""
    th = 2.0 * math.pi * j / n_poses
    c = np.asarray(centre, dtype=np.float64)
    pos = c + np.array([radius * math.cos(th), 0.0, radius * math.sin(th)])
    return look_at(pos, c)


# name -> parameters.  "uniform": config 1/2 distribution; "blobs": config 3/4/5 distribution.
CONFIGS: Dict[str, Dict] = {
    "cfg1": dict(kind="uniform", N=2_000, W=64, H=64, D=16, K=40, backward=False, feat_dtype="f32"),
    "cfg2": dict(kind="uniform", N=50_000, W=256, H=256, D=64, K=40, backward=True, feat_dtype="f32"),
    "cfg3": dict(kind="blobs", N=500_000, W=640, H=480, D=512, K=40, backward=True, feat_dtype="f32"),
    "cfg4": dict(kind="blobs", N=2_000_000, W=1024, H=768, D=512, K=32, backward=True, feat_dtype="f16",
                 pose=0, n_poses=8),
    "cfg5": dict(kind="blobs", N=1_000_000, W=1280, H=720, D=512, K=40, backward=True, feat_dtype="f32"),
}


def _unit_rows(a: np.ndarray) -> np.ndarray:
    n = np.sqrt((a.astype(np.float64) ** 2).sum(axis=1, keepdims=True))
    n[n == 0] = 1.0
    return (a / n).astype(np.float32)


def _log_uniform(rng, lo, hi, size):
    u = rng.random(size, dtype=np.float32)
    return np.exp(np.float32(math.log(lo)) + u * np.float32(math.log(hi) - math.log(lo))).astype(np.float32)


def make_scene(name: str = "cfg1", seed: int = 0, *, N: Optional[int] = None, W: Optional[int] = None,
               H: Optional[int] = None, D: Optional[int] = None, K: Optional[int] = None,
               backward: Optional[bool] = None, feat_dtype: Optional[str] = None,
               pose: Optional[int] = None, kind: Optional[str] = None) -> Scene:
    """Build one of the BASELINE.json configs; keyword overrides give scaled-down test variants
    with the same distributions (used by the parity tests at sizes the oracle finishes in seconds)."""
    p = dict(CONFIGS[name])
    for k, v in dict(N=N, W=W, H=H, D=D, K=K, backward=backward, feat_dtype=feat_dtype,
                     pose=pose, kind=kind).items():
        if v is not None:
            p[k] = v
    rng = np.random.default_rng(seed)
    n, d = int(p["N"]), int(p["D"])
    f32 = np.float32

    if p["kind"] == "uniform":
        means = np.empty((n, 3), dtype=f32)
        means[:, 0:2] = rng.random((n, 2), dtype=f32) * f32(2.0) - f32(1.0)
        means[:, 2] = rng.random(n, dtype=f32) * f32(4.0) + f32(2.0)
        scales = _log_uniform(rng, 0.01, 0.1, (n, 3))
        quats = _unit_rows(rng.standard_normal((n, 4), dtype=f32))
        opac = (rng.random(n, dtype=f32) * f32(0.94) + f32(0.05)).astype(f32)
        blob_of = None
        w2c = None
    elif p["kind"] == "blobs":
        n_blobs = 64
        half = np.array([4.0, 2.0, 4.0], dtype=f32)   # box 8 x 4 x 8 (x, y, z), centred at the origin
        centres = (rng.random((n_blobs, 3), dtype=f32) * f32(2.0) - f32(1.0)) * half
        blob_of = rng.integers(0, n_blobs, size=n)
        means = (centres[blob_of] + f32(0.3) * rng.standard_normal((n, 3), dtype=f32)).astype(f32)
        scales = _log_uniform(rng, 0.005, 0.05, (n, 3))
        quats = _unit_rows(rng.standard_normal((n, 4), dtype=f32))
        opac = rng.beta(2.0, 2.0, size=n).astype(f32)
        opac = np.clip(opac, f32(1e-4), f32(1.0 - 1e-4))
        w2c = pose_on_circle(int(p["pose"]), int(p.get("n_poses", 8))) if "pose" in p else None
    else:
        raise ValueError(p["kind"])

    cam = make_camera(int(p["W"]), int(p["H"]), 60.0, 0.2, w2c)

    # features are always drawn 512 wide when D <= 512 so that config 5's D sweep uses
    # "the first D columns of one 512-D draw, re-normalised".
    d_draw = max(d, 512) if p["kind"] == "blobs" else d
    if p["kind"] == "blobs":
        c_feat = _unit_rows(rng.standard_normal((64, d_draw), dtype=f32))
        feats = c_feat[blob_of]
        # add the noise in row chunks to bound peak memory at N = 2e6
        step = 65536
        for s in range(0, n, step):
            e = min(n, s + step)
            feats[s:e] += f32(0.1) * rng.standard_normal((e - s, d_draw), dtype=f32)
    else:
        feats = rng.standard_normal((n, d_draw), dtype=f32)
    feats = _unit_rows(np.ascontiguousarray(feats[:, :d]))

    fdt = p["feat_dtype"]
    if fdt == "f16":
        feats = feats.astype(np.float16)
    elif fdt != "f32":
        raise ValueError(fdt)

    dL = None
    if p["backward"]:
        dL = rng.standard_normal((cam.height, cam.width, d), dtype=f32)

    return Scene(name=name, cam=cam, means=np.ascontiguousarray(means), scales=scales,
                 quats=quats, opac=np.ascontiguousarray(opac), features=np.ascontiguousarray(feats),
                 dL_dmap=dL, K=int(p["K"]), feat_dtype=fdt, meta=dict(p, seed=seed))

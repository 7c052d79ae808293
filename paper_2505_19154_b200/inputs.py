"""Seeded synthetic inputs for the five BASELINE.json configs (SURVEY.md §8(d) generator table).

This module serves BOTH the CUDA path and the oracle and therefore holds none of the method's
arithmetic: it only draws random scenes, builds pinhole camera matrices and draws ground-truth
feature maps.  Everything is numpy on the host; the same arrays are handed to both sides.

Conventions:
  * world and camera are y-down, camera looks along +z; `view` is world->camera, row-major,
    applied to column vectors; `proj` is row-major with w_clip = z_cam and only entries
    [0],[2],[5],[6] meaningful: proj[0] = 2 fx / W, proj[5] = 2 fy / H,
    proj[2] = 2 (cx + 1/2) / W - 1, proj[6] = 2 (cy + 1/2) / H - 1.
  * `scale` and `opacity` are ACTIVATED (exp / sigmoid applied here once, on the host).
  * quaternion order (w, x, y, z).
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

SH_C0 = 0.28209479177387814  # only used to place the degree-0 coefficient so that colour = c


@dataclasses.dataclass
class Camera:
    view: np.ndarray      # [16] f32 row-major world->camera
    proj: np.ndarray      # [16] f32 row-major
    cam_pos: np.ndarray   # [3]  f32
    width: int
    height: int


@dataclasses.dataclass
class Scene:
    mean: np.ndarray      # [N,3] f32
    scale: np.ndarray     # [N,3] f32, > 0
    quat: np.ndarray      # [N,4] f32 (w,x,y,z)
    opacity: np.ndarray   # [N]   f32 in [0,1]
    sh: np.ndarray        # [N,K,3] f32, K=(deg+1)^2
    feat: np.ndarray      # [N,D] f32 or f16 ("bf16": f32 values that are exactly representable in bfloat16)
    sh_degree: int

    @property
    def n(self) -> int:
        return int(self.mean.shape[0])

    @property
    def feat_dim(self) -> int:
        return int(self.feat.shape[1])


@dataclasses.dataclass
class Config:
    name: str
    seed: int
    n: int
    feat_dim: int
    feat_dtype: str          # "f32" | "f16" | "bf16" (numpy has no bfloat16: values are rounded, the array stays f32)
    sh_degree: int
    width: int
    height: int
    n_views: int
    mean_half_extent: float
    log_scale_mu: float
    log_scale_sigma: float
    unit_features: bool
    gt_kind: str             # "normal" | "blurred" | "unit" | "blobs"


CONFIGS = {
    "tiny": Config("tiny", 1001, 1_000, 8, "f32", 0, 64, 64, 4, 1.0, -3.0, 0.5, False, "normal"),
    "small": Config("small", 1002, 100_000, 16, "f32", 1, 256, 256, 8, 2.0, -3.0, 0.5, False, "blurred"),
    "mid": Config("mid", 1003, 1_000_000, 128, "f32", 3, 1920, 1080, 1, 2.0, -4.0, 0.7, True, "unit"),
    "large": Config("large", 1004, 3_000_000, 512, "f16", 3, 1920, 1080, 1, 2.0, -4.0, 0.7, True, "unit"),
    "multiview": Config("multiview", 1005, 2_000_000, 256, "f32", 0, 1296, 968, 200, 5.0, -4.0, 0.7, True, "blobs"),
}


def round_to_bf16(a: np.ndarray) -> np.ndarray:
    """fp32 -> nearest bfloat16 (ties to even), returned as fp32: what a bf16 store of `a` holds.  Finite inputs."""
    u = np.ascontiguousarray(a, dtype=np.float32).view(np.uint32)
    r = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + r) & np.uint32(0xFFFF0000)).view(np.float32)


def scaled(cfg: Config, **kw) -> Config:
    """A copy of `cfg` with some fields replaced (used for reduced-size parity cases)."""
    return dataclasses.replace(cfg, **kw)


# ----------------------------------------------------------------------------------------------
# cameras
# ----------------------------------------------------------------------------------------------
def look_at_camera(pos, target, width: int, height: int, fov_x_deg: float = 60.0,
                   down=(0.0, 1.0, 0.0)) -> Camera:
    """Pinhole camera at `pos` looking at `target`; camera +y follows world `down`."""
    pos = np.asarray(pos, dtype=np.float64)
    target = np.asarray(target, dtype=np.float64)
    f = target - pos
    f = f / np.linalg.norm(f)
    d0 = np.asarray(down, dtype=np.float64)
    r = np.cross(d0, f)
    r = r / np.linalg.norm(r)
    d = np.cross(f, r)
    rot = np.stack([r, d, f], axis=0)            # rows = camera axes in world coordinates
    view = np.eye(4)
    view[:3, :3] = rot
    view[:3, 3] = -rot @ pos
    fx = (width / 2.0) / math.tan(math.radians(fov_x_deg) / 2.0)
    fy = fx                                       # square pixels
    cx = (width - 1) / 2.0
    cy = (height - 1) / 2.0
    proj = np.zeros((4, 4))
    proj[0, 0] = 2.0 * fx / width
    proj[1, 1] = 2.0 * fy / height
    proj[0, 2] = 2.0 * (cx + 0.5) / width - 1.0
    proj[1, 2] = 2.0 * (cy + 0.5) / height - 1.0
    proj[2, 2] = 1.0
    proj[3, 2] = 1.0                              # w_clip = z_cam
    return Camera(view.astype(np.float32).reshape(16), proj.astype(np.float32).reshape(16),
                  pos.astype(np.float32), int(width), int(height))


def circle_camera(k: int, n_views: int, width: int, height: int, radius: float = 4.0) -> Camera:
    th = 2.0 * math.pi * k / n_views
    pos = (radius * math.sin(th), 0.0, -radius * math.cos(th))
    return look_at_camera(pos, (0.0, 0.0, 0.0), width, height)


def orbit_camera(v: int, cfg: Config) -> Camera:
    """Multi-view 'jittered orbit' camera v (SURVEY §8(d) reading)."""
    rng = np.random.default_rng(cfg.seed * 1000 + 500 + v)
    th = 2.0 * math.pi * v / cfg.n_views
    radius = 4.5 + rng.uniform(-0.25, 0.25)
    height = rng.uniform(-0.5, 0.5)
    target = rng.uniform(-0.5, 0.5, size=3)
    pos = (radius * math.sin(th), height, -radius * math.cos(th))
    return look_at_camera(pos, target, cfg.width, cfg.height)


def crop_camera(cam: Camera, x0: int, y0: int, width: int, height: int) -> Camera:
    """The same pinhole camera restricted to the pixel window [x0,x0+width) x [y0,y0+height): fx, fy
    and the view matrix are unchanged, the principal point moves by (-x0,-y0).  Pure camera
    bookkeeping (used for bounded oracle samples of a large frame)."""
    w, h = cam.width, cam.height
    proj = cam.proj.astype(np.float64).reshape(4, 4).copy()
    fx = proj[0, 0] * w / 2.0
    fy = proj[1, 1] * h / 2.0
    cx = (proj[0, 2] + 1.0) * w / 2.0 - 0.5 - x0
    cy = (proj[1, 2] + 1.0) * h / 2.0 - 0.5 - y0
    proj[0, 0] = 2.0 * fx / width
    proj[1, 1] = 2.0 * fy / height
    proj[0, 2] = 2.0 * (cx + 0.5) / width - 1.0
    proj[1, 2] = 2.0 * (cy + 0.5) / height - 1.0
    return Camera(cam.view.copy(), proj.astype(np.float32).reshape(16), cam.cam_pos.copy(), int(width), int(height))


def make_camera(cfg: Config, view_idx: int) -> Camera:
    if cfg.gt_kind == "blobs":
        return orbit_camera(view_idx, cfg)
    return circle_camera(view_idx, cfg.n_views, cfg.width, cfg.height)


# ----------------------------------------------------------------------------------------------
# scenes
# ----------------------------------------------------------------------------------------------
def _unit_rows(a: np.ndarray) -> np.ndarray:
    nrm = np.sqrt((a.astype(np.float64) ** 2).sum(axis=1, keepdims=True))
    return (a / np.maximum(nrm, 1e-30)).astype(np.float32)


def blob_centres(cfg: Config) -> np.ndarray:
    rng = np.random.default_rng(cfg.seed + 70_000)
    return rng.uniform(-4.0, 4.0, size=(64, 3))


def blob_vectors(cfg: Config) -> np.ndarray:
    """65 random unit vectors: 64 blob features + 1 background (row 64)."""
    rng = np.random.default_rng(cfg.seed + 80_000)
    return _unit_rows(rng.standard_normal((65, cfg.feat_dim)))


def make_scene(cfg: Config) -> Scene:
    rng = np.random.default_rng(cfg.seed)
    n = cfg.n
    if cfg.gt_kind == "blobs":
        centres = blob_centres(cfg)
        owner = np.arange(n) % 64
        mean = (centres[owner] + 0.3 * rng.standard_normal((n, 3))).astype(np.float32)
    else:
        mean = rng.uniform(-cfg.mean_half_extent, cfg.mean_half_extent, size=(n, 3)).astype(np.float32)
    scale = np.exp(cfg.log_scale_mu + cfg.log_scale_sigma * rng.standard_normal((n, 3))).astype(np.float32)
    quat = _unit_rows(rng.standard_normal((n, 4)))
    opacity = (1.0 / (1.0 + np.exp(-rng.standard_normal(n)))).astype(np.float32)
    k = (cfg.sh_degree + 1) ** 2
    sh = np.empty((n, k, 3), dtype=np.float32)
    colour = rng.uniform(0.0, 1.0, size=(n, 3))
    sh[:, 0, :] = ((colour - 0.5) / SH_C0).astype(np.float32)
    if k > 1:
        sh[:, 1:, :] = (0.1 * rng.standard_normal((n, k - 1, 3), dtype=np.float32))
    feat = rng.standard_normal((n, cfg.feat_dim), dtype=np.float32)
    if cfg.unit_features:
        feat = _unit_rows(feat)
    if cfg.feat_dtype == "f16":
        feat = feat.astype(np.float16)
    elif cfg.feat_dtype == "bf16":
        feat = round_to_bf16(feat)
    return Scene(mean, scale, quat, opacity, sh, feat, cfg.sh_degree)


# ----------------------------------------------------------------------------------------------
# ground-truth feature maps
# ----------------------------------------------------------------------------------------------
def _blur_axis(a: np.ndarray, axis: int, sigma: float, radius: int) -> np.ndarray:
    xs = np.arange(-radius, radius + 1)
    kern = np.exp(-0.5 * (xs / sigma) ** 2)
    kern = kern / kern.sum()
    n = a.shape[axis]
    out = np.zeros_like(a, dtype=np.float64)
    idx = np.arange(n)
    for j, wgt in zip(xs, kern):
        src = np.clip(idx + j, 0, n - 1)          # edge-clamped
        out += wgt * np.take(a, src, axis=axis)
    return out


def make_gt_map(cfg: Config, view_idx: int, cam: Camera | None = None) -> np.ndarray:
    """[H,W,D] ground-truth feature map for one view (dtype follows cfg.feat_dtype)."""
    h, w, d = cfg.height, cfg.width, cfg.feat_dim
    rng = np.random.default_rng(cfg.seed * 1000 + view_idx)
    if cfg.gt_kind == "normal":
        g = rng.standard_normal((h, w, d), dtype=np.float32)
    elif cfg.gt_kind == "blurred":
        g = rng.standard_normal((h, w, d))
        g = _blur_axis(_blur_axis(g, 0, 2.0, 6), 1, 2.0, 6).astype(np.float32)
    elif cfg.gt_kind == "unit":
        g = rng.standard_normal((h, w, d), dtype=np.float32)
        nrm = np.sqrt(np.einsum("hwd,hwd->hw", g, g, dtype=np.float32))[..., None]
        g /= np.maximum(nrm, 1e-30)
    elif cfg.gt_kind == "blobs":
        cam = cam or make_camera(cfg, view_idx)
        label = blob_label_map(cfg, cam)
        vecs = blob_vectors(cfg)
        g = vecs[label] + 0.05 * rng.standard_normal((h, w, d), dtype=np.float32)
        g = g.astype(np.float32)
    else:
        raise ValueError(cfg.gt_kind)
    if cfg.feat_dtype == "f16":
        g = g.astype(np.float16)
    elif cfg.feat_dtype == "bf16":
        g = round_to_bf16(g)
    return np.ascontiguousarray(g)


def make_gt_map_blobs_torch(cfg: Config, view_idx: int, cam: Camera, device, out=None):
    """The Multi-view config's per-view map built ON THE DEVICE (1.28 GB each, 257 GB for the 200 views:
    generated per view, seeded `cfg.seed * 1000 + view_idx`, never all resident): the same recipe as make_gt_map's
    "blobs" branch -- label map from the pinhole rays (host, 64 blobs), blob vector + N(0, 0.05^2) noise drawn by torch's
    generator.  The values differ from make_gt_map's numpy draws (another generator); the parity tests use make_gt_map
    on both sides, the 200-view sweep uses this one and is checked through invariants."""
    import torch
    assert cfg.gt_kind == "blobs"
    label = torch.from_numpy(blob_label_map(cfg, cam)).to(device)
    vecs = torch.from_numpy(blob_vectors(cfg).astype(np.float32)).to(device)
    gen = torch.Generator(device=device).manual_seed(cfg.seed * 1000 + view_idx)
    if out is None:
        out = torch.empty((cfg.height, cfg.width, cfg.feat_dim), dtype=torch.float32, device=device)
    out.normal_(0.0, 0.05, generator=gen)
    out += vecs[label]
    return out


def blob_label_map(cfg: Config, cam: Camera) -> np.ndarray:
    """[H,W] int: index of the nearest blob along the pixel ray whose centre lies within 0.6 of
    the ray, else 64 (background).  Pure input geometry (pinhole rays), not the splatting method."""
    h, w = cam.height, cam.width
    view = cam.view.astype(np.float64).reshape(4, 4)
    proj = cam.proj.astype(np.float64)
    fx = proj[0] * w / 2.0
    fy = proj[5] * h / 2.0
    cx = (proj[2] + 1.0) * w / 2.0 - 0.5
    cy = (proj[6] + 1.0) * h / 2.0 - 0.5
    c = blob_centres(cfg)
    cc = (view[:3, :3] @ c.T).T + view[:3, 3]     # [64,3] camera frame
    xs = (np.arange(w) - cx) / fx
    ys = (np.arange(h) - cy) / fy
    dirs = np.stack(np.broadcast_arrays(xs[None, :], ys[:, None], 1.0), axis=-1)
    dirs = dirs / np.linalg.norm(dirs, axis=-1, keepdims=True)      # [H,W,3]
    best_t = np.full((h, w), np.inf)
    label = np.full((h, w), 64, dtype=np.int64)
    for j in range(64):
        t = dirs @ cc[j]                          # distance along the ray of the closest approach
        d2 = (cc[j] ** 2).sum() - t * t
        hit = (t > 0.2) & (d2 <= 0.36) & (t < best_t)
        best_t = np.where(hit, t, best_t)
        label = np.where(hit, j, label)
    return label

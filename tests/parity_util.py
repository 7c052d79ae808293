"""Shared helpers of the GPU parity tests (and of __graft_entry__.smoke()): run the CUDA path through
the C ABI binding and the CPU oracle on the same seeded inputs, and compare per the rules of
SURVEY.md 8(c) / DESIGN.md "Tolerances".  Test infrastructure: may import oracle/."""
from __future__ import annotations

import numpy as np

from oracle import fhgs_oracle as fo
from paper_2505_19154_b200 import inputs

TOL_F32 = 1e-4      # north_star: max abs on fp32 RGB, features and fused vectors
TOL_F16 = 2e-3      # north_star: where features are stored fp16


def cam35(cam):
    return fo.cam_array(cam.view, cam.proj, cam.cam_pos)


def oracle_view(scene, cam, params=fo.DEFAULT_PARAMS):
    pr = fo.project(scene.mean, scene.scale, scene.quat, scene.opacity, scene.sh, scene.sh_degree, cam35(cam),
                    cam.width, cam.height, params)
    return pr


class GpuPath:
    """One scene on the device + a reusable view state."""

    def __init__(self, scene, width, height, capacity, device=0):
        import torch
        from paper_2505_19154_b200 import binding as fb
        self.torch, self.fb = torch, fb
        self.ctx = fb.Context(device)
        self.g = fb.Gaussians(scene.mean, scene.scale, scene.quat, scene.opacity, scene.sh, scene.feat, scene.sh_degree)
        self.vs = fb.ViewState(scene.n, width, height, capacity)
        self.prm = fb.default_params()
        self.W, self.H = width, height
        self.D = scene.feat_dim

    def camera(self, cam):
        return self.fb.make_camera(cam.view, cam.proj, cam.cam_pos, cam.width, cam.height)

    def project_sort(self, cam, flags=0):
        c = self.camera(cam)
        self.fb.project(self.ctx, self.g, c, self.prm, self.vs)
        m = self.fb.bin_sort(self.ctx, c, self.vs, sync=True, flags=flags)
        return c, m

    def render(self, c, with_feat=True):
        t = self.torch
        dev = self.g.mean.device
        out = dict(rgb=t.empty((self.H, self.W, 3), dtype=t.float32, device=dev),
                   T=t.empty((self.H, self.W), dtype=t.float32, device=dev),
                   n=t.empty((self.H, self.W), dtype=t.int32, device=dev),
                   feat=t.empty((self.H, self.W, self.D), dtype=self.g.feat.dtype, device=dev) if with_feat else None)
        self.fb.render(self.ctx, self.g, c, self.prm, self.vs, out["rgb"], out["feat"], out["T"], out["n"])
        t.cuda.synchronize()
        return {k: (None if v is None else v.cpu().numpy()) for k, v in out.items()}

    def fuse(self, c, gt, num=None, den=None, flags=None, out_dtype=None):
        t, fb = self.torch, self.fb
        dev = self.g.mean.device
        n = self.g.n
        gt_d = t.from_numpy(np.ascontiguousarray(gt)).to(dev)
        if num is None:
            num = t.zeros((n, self.D), dtype=t.float32, device=dev)
            den = t.zeros((n,), dtype=t.float32, device=dev)
        fl = fb.FHGS_FUSE_ZERO if flags is None else flags
        fb.fuse_features(self.ctx, c, self.prm, self.vs, gt_d, num, den, None, fl)
        t.cuda.synchronize()
        return num, den

    def finalize(self, num, den, prev, l2norm=False):
        t, fb = self.torch, self.fb
        out = t.from_numpy(np.ascontiguousarray(prev)).to(num.device)
        fl = fb.FHGS_FUSE_FINALIZE_ONLY | (fb.FHGS_FUSE_L2NORM if l2norm else 0)
        fb.fuse_features(self.ctx, None, self.prm, self.vs, None, num, den, out, fl)
        t.cuda.synchronize()
        return out.cpu().numpy()


def check_projection(pr_o, pr_g):
    """Integer outputs bit-exact; float outputs bit-exact by construction (C1-P), rgb within 1e-4."""
    for k in ("radius", "rect", "tiles_touched"):
        assert np.array_equal(pr_o[k], pr_g[k]), f"projection integer output {k} differs"
    for k in ("xy", "depth", "conic_opacity"):
        assert np.array_equal(pr_o[k].view(np.uint32), pr_g[k].view(np.uint32)), f"projection float output {k} not bit-equal"
    assert np.max(np.abs(pr_o["rgb"] - pr_g["rgb"]), initial=0.0) <= TOL_F32


def check_bins(bo, vs, m):
    assert m == bo["M"], f"M differs: gpu {m} oracle {bo['M']}"
    n = bo["offsets"].shape[0]
    assert np.array_equal(vs.offsets[:n].cpu().numpy().view(np.uint32), bo["offsets"])
    assert np.array_equal(vs.sorted_keys(m), bo["keys"]), "sorted keys differ"
    assert np.array_equal(vs.sorted_vals(m), bo["vals"]), "sorted values differ"
    assert np.array_equal(vs.ranges.cpu().numpy().view(np.uint32), bo["ranges"]), "tile ranges differ"


def check_render(o, g, feat_absmax, tol, pix=None, with_feat=True):
    """o: oracle dict (npix rows); g: GPU dict of full images; pix: linear pixel ids of o's rows."""
    H, W = g["T"].shape
    sel = np.arange(H * W) if pix is None else np.asarray(pix)
    frag = o["fragile"].astype(bool)
    n_g = g["n"].reshape(-1)[sel].view(np.uint32).astype(np.int64)
    dn = np.abs(n_g - o["n"].astype(np.int64))
    assert np.all(dn[~frag] == 0), f"n_contrib differs on {int((dn[~frag] != 0).sum())} non-fragile pixels"
    assert np.all(dn[frag] <= 1), "n_contrib differs by more than 1 on a fragile pixel"
    slack = np.where(frag, tol + 1e-4 * max(feat_absmax, 1.0), tol)
    d_rgb = np.abs(g["rgb"].reshape(-1, 3)[sel] - o["rgb"]).max(axis=1)
    assert np.all(d_rgb <= slack), f"rgb max abs err {d_rgb.max():.3e}"
    d_T = np.abs(g["T"].reshape(-1)[sel] - o["T"])
    assert np.all(d_T <= slack), f"T max abs err {d_T.max():.3e}"
    worst = dict(rgb=float(d_rgb.max(initial=0)), T=float(d_T.max(initial=0)), fragile=int(frag.sum()))
    if with_feat:
        D = g["feat"].shape[-1]
        d_f = np.abs(g["feat"].reshape(-1, D)[sel].astype(np.float64) - o["feat"]).max(axis=1)
        assert np.all(d_f <= slack), f"feature image max abs err {d_f.max():.3e} (tol {tol})"
        worst["feat"] = float(d_f.max(initial=0))
    return worst


def gaussians_touching(pr, pix, W):
    """Per Gaussian, the number of the given pixels that lie inside its radius box."""
    touched = np.zeros(pr["radius"].shape[0], np.int64)
    r = pr["radius"].astype(np.float32)
    vis = r > 0
    for p in np.asarray(pix):
        x, y = float(p % W), float(p // W)
        touched += vis & (np.abs(pr["xy"][:, 0] - x) <= r) & (np.abs(pr["xy"][:, 1] - y) <= r)
    return touched


def check_fuse(num_o, den_o, num_g, den_g, gt_absmax, tol, fragile_touch=None):
    """num/den: |d den| <= tol*max(den,1), |d num| <= tol*max(den,1)*|G|max; Gaussians touching a fragile
    pixel get the extra 1e-4 per fragile pixel that one borderline contributor may add or drop."""
    num_g = num_g.cpu().numpy().astype(np.float64)
    den_g = den_g.cpu().numpy().astype(np.float64)
    scale = np.maximum(den_o, 1.0)
    extra = np.zeros_like(den_o) if fragile_touch is None else fragile_touch.astype(np.float64) * 1.1e-4
    d_den = np.abs(den_g - den_o)
    assert np.all(d_den <= tol * scale + extra), f"den max err {d_den.max():.3e}"
    d_num = np.abs(num_g - num_o).max(axis=1)
    assert np.all(d_num <= (tol * scale + extra) * max(gt_absmax, 1.0)), f"num max err {d_num.max():.3e}"
    return dict(den=float(d_den.max(initial=0)), num=float(d_num.max(initial=0)))


def check_finalized(f_o, f_g, den_o, tol, den_floor=1e-3, fragile_mask=None):
    """Finalised vectors within tol for every Gaussian with den >= den_floor that touches no fragile pixel
    (below the floor one borderline weight of 1e-4 legitimately moves the mean)."""
    sel = den_o >= den_floor
    if fragile_mask is not None:
        sel &= ~(fragile_mask.astype(bool))
    d = np.abs(f_g.astype(np.float64)[sel] - f_o[sel])
    assert d.size == 0 or d.max() <= tol, f"fused feature max abs err {d.max():.3e} (tol {tol})"
    return float(d.max(initial=0)), int(sel.sum())


def reduced_config(name, **kw):
    return inputs.scaled(inputs.CONFIGS[name], **kw)

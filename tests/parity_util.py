"""Shared helpers of the GPU parity tests (and of __graft_entry__.smoke()): run the CUDA path through
the C ABI binding and the CPU oracle on the same seeded inputs, and compare per the rules of
SURVEY.md 8(c) / DESIGN.md "Tolerances".  Test infrastructure: may import oracle/."""
from __future__ import annotations

import numpy as np

from oracle import fhgs_oracle as fo
from paper_2505_19154_b200 import inputs

TOL_F32 = 1e-4      # north_star: max abs on fp32 RGB, features and fused vectors
TOL_F16 = 2e-3      # north_star: where features are stored fp16
# bf16 storage (NEXT-4 iv; north_star states no bar): one rounding to 8 significant bits of an output of magnitude <= 1
# is <= 2^-9 = 1.95e-3, on top of the fp32 accumulation bound 1e-4 ("Tolerances")
TOL_BF16 = 2.5e-3


def cam35(cam):
    return fo.cam_array(cam.view, cam.proj, cam.cam_pos)


def oracle_view(scene, cam, params=fo.DEFAULT_PARAMS):
    pr = fo.project(scene.mean, scene.scale, scene.quat, scene.opacity, scene.sh, scene.sh_degree, cam35(cam),
                    cam.width, cam.height, params)
    return pr


class GpuPath:
    """One scene on the device + a reusable view state."""

    def __init__(self, scene, width, height, capacity, device=0, surfel=False, storage=None):
        """storage="bf16": feature rows, GT maps and feature outputs are stored as bfloat16 on the device (the numpy
        arrays carry bf16-exact f32 values); results come back widened to f32."""
        import torch
        from paper_2505_19154_b200 import binding as fb
        self.torch, self.fb = torch, fb
        self.ctx = fb.Context(device)
        self.bf16 = storage == "bf16"
        feat = torch.from_numpy(np.ascontiguousarray(scene.feat)).to(torch.bfloat16) if self.bf16 else scene.feat
        self.g = fb.Gaussians(scene.mean, scene.scale, scene.quat, scene.opacity, scene.sh, feat, scene.sh_degree)
        self.vs = fb.ViewState(scene.n, width, height, capacity, surfel=surfel)
        self.prm = fb.default_params(primitive=fb.FHGS_PRIM_SURFEL if surfel else fb.FHGS_PRIM_EWA)
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
        return {k: (None if v is None else (v.float() if v.dtype == t.bfloat16 else v).cpu().numpy()) for k, v in out.items()}

    def fuse(self, c, gt, num=None, den=None, flags=None, out_dtype=None):
        t, fb = self.torch, self.fb
        dev = self.g.mean.device
        n = self.g.n
        gt_d = t.from_numpy(np.ascontiguousarray(gt)).to(dev)
        if self.bf16:
            gt_d = gt_d.to(t.bfloat16)   # exact: the map holds bf16-representable values
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
        if self.bf16:
            out = out.to(t.bfloat16)
        fl = fb.FHGS_FUSE_FINALIZE_ONLY | (fb.FHGS_FUSE_L2NORM if l2norm else 0)
        fb.fuse_features(self.ctx, None, self.prm, self.vs, None, num, den, out, fl)
        t.cuda.synchronize()
        return (out.float() if self.bf16 else out).cpu().numpy()


def check_projection(pr_o, pr_g):
    """Integer outputs bit-exact; float outputs bit-exact by construction (C1-P), rgb within 1e-4."""
    for k in ("radius", "rect", "tiles_touched"):
        assert np.array_equal(pr_o[k], pr_g[k]), f"projection integer output {k} differs"
    for k in ("xy", "depth", "conic_opacity") + (("ray_transform",) if "ray_transform" in pr_o else ()):
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


class Borderline:
    """Borderline fragments of a set of views: fragments whose incoming transmittance T lies within `window`
    (relative) of t_min, so that the stop test `T < t_min` may legitimately come out differently on the two sides
    (exp differs by a few ulp between them).  Fragments in front of them are blended by both sides, fragments behind
    them by neither.  For each: Gaussian index, weight w = alpha*T, whether the ORACLE blended it, and the GT row of
    its pixel.  Where several results are correct the tests accept each of them -- and nothing else."""

    def __init__(self, n, D):
        self.n, self.D = n, D
        self.g, self.w, self.blended, self.G = [], [], [], []

    def add_view(self, pr, pix, W, bins, gt, q_cutoff=9.0, alpha_max=0.9999, t_min=1e-4, window=2e-4):
        """pix: the view's fragile pixels (oracle flag).  The pixel's fragment sequence is rebuilt from the oracle's
        projection and its sorted tile list `bins` (fo.bins): binary32 q as C1-R states it, then double."""
        f32, f64 = np.float32, np.float64
        gx, gy = pr["xy"][:, 0], pr["xy"][:, 1]
        co = pr["conic_opacity"]
        GW = (W + 15) // 16
        gt2 = gt.reshape(-1, gt.shape[-1])
        for p in np.asarray(pix):
            x, y = int(p % W), int(p // W)
            r0, r1 = bins["ranges"][(y // 16) * GW + x // 16]
            cand = bins["vals"][int(r0):int(r1)].astype(np.int64)          # front to back
            if cand.size == 0:
                continue
            if "ray_transform" in pr:   # surfel mode: u^2 + v^2 from the ray transform (the cut-off edge itself is not at stake here)
                rt = pr["ray_transform"][cand].astype(f64)
                p0, p1, p2 = (x * rt[:, 4 * r] + y * rt[:, 4 * r + 1] + rt[:, 4 * r + 2] for r in range(3))
                num, den = p0 * p0 + p1 * p1, p2 * p2
                c = (den > 0) & (num <= q_cutoff * den)
                q = np.where(c, num / np.where(den > 0, den, 1.0), 0.0)
            else:
                dx, dy = (gx[cand] - f32(x)).astype(f32), (gy[cand] - f32(y)).astype(f32)
                A, B2, Cc = co[cand, 0], (f32(2.0) * co[cand, 1]).astype(f32), co[cand, 2]
                adx = (A * dx).astype(f32)
                inner = (B2.astype(f64) * dy.astype(f64) + adx.astype(f64)).astype(f32)          # fmaf(2B, dy, A dx)
                cdy2 = ((Cc * dy).astype(f32) * dy).astype(f32)
                q = (dx.astype(f64) * inner.astype(f64) + cdy2.astype(f64)).astype(f32)          # fmaf(dx, inner, (C dy) dy)
                c = q <= f32(q_cutoff)
            alpha = np.where(c, np.minimum(f64(f32(alpha_max)), co[cand, 3].astype(f64) * np.exp(-0.5 * np.maximum(q.astype(f64), 0.0))), 0.0)
            T_before = np.concatenate([[1.0], np.cumprod(1.0 - alpha)[:-1]])
            for j in np.nonzero(c & (np.abs(T_before / t_min - 1.0) <= window))[0]:
                self.g.append(int(cand[j])); self.w.append(float(alpha[j] * T_before[j]))
                self.blended.append(bool(T_before[j] >= t_min)); self.G.append(gt2[p].astype(f64))

    def weight_mass(self):
        """Per Gaussian, the total weight of its borderline fragments."""
        m = np.zeros(self.n)
        if self.g:
            np.add.at(m, np.asarray(self.g), np.asarray(self.w))
        return m

    def by_gaussian(self):
        out = {}
        for j, g in enumerate(self.g):
            out.setdefault(g, []).append(j)
        return out


def check_fuse(num_o, den_o, num_g, den_g, gt_absmax, tol, border=None):
    """Accumulators, RELATIVE to the row's own weight mass (no absolute floor):
        |d den_i| <= tol den_i + b_i,   |d num_i|max <= (tol den_i + b_i) |G|max
    with b_i = 1.01 x the weight mass of Gaussian i's borderline fragments (0 for almost every row).  A row the oracle
    never blends (den_i = 0) must therefore be exactly zero on the GPU unless it has a borderline fragment."""
    num_g = num_g.cpu().numpy().astype(np.float64)
    den_g = den_g.cpu().numpy().astype(np.float64)
    b = np.zeros_like(den_o) if border is None else 1.01 * border.weight_mass()
    bound = tol * den_o + b
    d_den = np.abs(den_g - den_o)
    bad = d_den > bound
    assert not bad.any(), f"den: {int(bad.sum())} rows off, worst {d_den[bad].max():.3e} at den {den_o[bad][np.argmax(d_den[bad])]:.3e}"
    d_num = np.abs(num_g - num_o).max(axis=1)
    bad = d_num > bound * max(gt_absmax, 1.0)
    assert not bad.any(), f"num: {int(bad.sum())} rows off, worst {d_num[bad].max():.3e}"
    live = den_o > 0
    rel = float((d_den[live] / den_o[live]).max(initial=0.0))
    return dict(den=float(d_den.max(initial=0)), num=float(d_num.max(initial=0)), den_rel=rel)


def check_finalized(f_o, f_g, prev, num_o, den_o, den_g, tol, den_eps=1e-8, border=None, max_alt=10):
    """Finalised vectors of EVERY row, no floor on den.  f_o: the oracle's finalised table (prev where not finalised).
    Rows without borderline fragments: finalised on both sides (den > den_eps; a den within a factor 2 of den_eps may
    be finalised on one side only and is skipped) and |f_g - f_o|max <= tol, or untouched on both sides.
    Rows WITH borderline fragments have several correct results: each subset of these fragments blended / not
    blended gives one (num', den') and f' = num'/den' (or the previous row when den' <= den_eps); f_g must be
    within tol of one of them.  Returns (worst error over all rows, rows finalised, rows resolved through an
    alternative, rows with more than `max_alt` borderline fragments = unchecked; the last must be 0)."""
    f_g = f_g.astype(np.float64)
    prev = np.asarray(prev, np.float64)
    den_g = np.asarray(den_g, np.float64)
    d = np.abs(f_g - f_o).max(axis=1)
    frag_rows = border.by_gaussian() if border is not None else {}
    has_frag = np.zeros(den_o.shape[0], bool)
    if frag_rows:
        has_frag[np.fromiter(frag_rows.keys(), np.int64)] = True
    fin_o, fin_g = den_o > den_eps, den_g > den_eps
    ambiguous = (den_o > 0.5 * den_eps) & (den_o < 2.0 * den_eps)
    plain = ~has_frag & ~ambiguous
    assert np.array_equal(fin_o[plain], fin_g[plain]), "a row is finalised on one side only"
    bad = plain & (d > tol)
    assert not bad.any(), (f"fused feature: {int(bad.sum())} rows off, worst {d[bad].max():.3e} (tol {tol}) at den "
                           f"{den_o[bad][np.argmax(d[bad])]:.3e}")
    worst = float(d[plain].max(initial=0))
    n_alt = n_unchecked = 0
    for g, idx in frag_rows.items():
        if d[g] <= tol and fin_o[g] == fin_g[g]:
            continue
        if len(idx) > max_alt:
            n_unchecked += 1
            continue
        n_alt += 1
        best = np.inf
        for mask in range(1 << len(idx)):
            num_a, den_a = num_o[g].copy(), den_o[g]
            for b, j in enumerate(idx):
                if mask >> b & 1:       # flip fragment j: remove it if the oracle blended it, else add it
                    sgn = -1.0 if border.blended[j] else 1.0
                    num_a += sgn * border.w[j] * border.G[j]
                    den_a += sgn * border.w[j]
            f_a = num_a / den_a if den_a > den_eps else prev[g]
            best = min(best, float(np.abs(f_g[g] - f_a).max()))
        assert best <= tol, f"fused feature of Gaussian {g}: no valid alternative within tol (best {best:.3e}, den {den_o[g]:.3e})"
        worst = max(worst, best)
    assert n_unchecked == 0, f"{n_unchecked} rows with more than {max_alt} borderline fragments"
    return worst, int(fin_o.sum()), n_alt, n_unchecked


def reduced_config(name, **kw):
    return inputs.scaled(inputs.CONFIGS[name], **kw)

"""Memory-safety checks of our own for every kernel variant (compute-sanitizer is closed on this GPU pool; see
profiles/r02_sanitizer.md).  Three instruments, all through the C ABI:

  * guard bands   every buffer the library may write (view state, scratch, key/value ping-pong, images, accumulators)
                  sits between two 4 KiB bands of a byte pattern; any band that changes is an out-of-bounds write.
  * poison        before each call the writable buffers are filled with garbage (0xFF.. = NaN / huge integers); the
                  results must still match the oracle bit for bit / within tolerance, so no kernel reads memory that
                  the path itself did not initialise (an initcheck stand-in), and every output element is written.
  * repetition    the whole sequence runs three times on the same poisoned buffers: P, S, R must repeat bit for bit
                  (a shared-memory race or a missing barrier shows up as run-to-run differences).
"""
import numpy as np
import pytest

from oracle import fhgs_oracle as fo
from paper_2505_19154_b200 import inputs
import parity_util as pu

pytestmark = pytest.mark.gpu

GUARD = 4096
PATTERN = 0xA5


class Guarded:
    """A device byte buffer with guard bands; .ptr is the 4096-aligned interior."""

    def __init__(self, torch, nbytes, dev):
        self.torch = torch
        self.nbytes = int(nbytes)
        self.raw = torch.full((self.nbytes + 2 * GUARD + 4096,), PATTERN, dtype=torch.uint8, device=dev)
        base = self.raw.data_ptr()
        self.off = (-(base + GUARD)) % 4096 + GUARD
        self.ptr = base + self.off
        self.poison()

    def interior(self):
        return self.raw[self.off:self.off + self.nbytes]

    def poison(self, value=0xFF):
        self.interior().fill_(value)

    def zero(self):
        self.interior().zero_()

    def intact(self):
        lo = self.raw[:self.off]
        hi = self.raw[self.off + self.nbytes:]
        return bool((lo == PATTERN).all().item()) and bool((hi == PATTERN).all().item())

    def view(self, dtype, shape):
        return self.interior().view(dtype).view(*shape)


def guarded_view_state(fb, torch, n, W, H, cap, dev, surfel=False):
    vs = fb.ViewState(n, W, H, cap, device=dev, surfel=surfel)
    gw, gh = (W + 15) // 16, (H + 15) // 16
    m, c = max(n, 1), max(cap, 1)
    sizes = dict(xy=8 * m, depth=4 * m, conic_opacity=16 * m, rgb=12 * m, radius=4 * m, rect=8 * m, tiles_touched=4 * m,
                 offsets=4 * m, num_instances=8, ranges=8 * gw * gh, scratch=int(vs.c.scratch_bytes),
                 keys0=8 * c, keys1=8 * c, vals0=4 * c, vals1=4 * c)
    if surfel:
        sizes["ray_transform"] = 48 * m
    bufs = {k: Guarded(torch, v, dev) for k, v in sizes.items()}
    if surfel:
        vs.c.ray_transform = bufs["ray_transform"].ptr
        vs.ray_transform = bufs["ray_transform"].view(torch.float32, (m, 12))
    for k in ("xy", "depth", "conic_opacity", "rgb", "radius", "rect", "tiles_touched", "offsets", "num_instances", "ranges", "scratch"):
        setattr(vs.c, k, bufs[k].ptr)
    vs.c.keys[0], vs.c.keys[1] = bufs["keys0"].ptr, bufs["keys1"].ptr
    vs.c.vals[0], vs.c.vals[1] = bufs["vals0"].ptr, bufs["vals1"].ptr
    # typed views for the comparisons (replace the binding's own tensors)
    vs.xy, vs.depth = bufs["xy"].view(torch.float32, (m, 2)), bufs["depth"].view(torch.float32, (m,))
    vs.conic_opacity, vs.rgb = bufs["conic_opacity"].view(torch.float32, (m, 4)), bufs["rgb"].view(torch.float32, (m, 3))
    vs.radius, vs.rect = bufs["radius"].view(torch.int32, (m,)), bufs["rect"].view(torch.int16, (m, 4))
    vs.tiles_touched, vs.offsets = bufs["tiles_touched"].view(torch.int32, (m,)), bufs["offsets"].view(torch.int32, (m,))
    vs.num_instances = bufs["num_instances"].view(torch.int64, (1,))
    vs.ranges = bufs["ranges"].view(torch.int32, (gw * gh, 2))
    vs.keys = [bufs["keys0"].view(torch.int64, (c,)), bufs["keys1"].view(torch.int64, (c,))]
    vs.vals = [bufs["vals0"].view(torch.int32, (c,)), bufs["vals1"].view(torch.int32, (c,))]
    vs.scratch = bufs["scratch"].interior()
    return vs, bufs


def run_guarded(cfg, view, tol, sort_flags=(1, 0), ndfd=False, surfel=False):
    import torch
    from paper_2505_19154_b200 import binding as fb
    scene = inputs.make_scene(cfg)
    cam = inputs.make_camera(cfg, view)
    gt = inputs.make_gt_map(cfg, view, cam)
    pr = pu.oracle_view(scene, cam, fo.params(primitive=1 if surfel else 0))
    bo = fo.bins(pr, cfg.width, cfg.height)
    order = fo.global_order(pr)
    feat32 = scene.feat.astype(np.float32)
    o = fo.render_scatter(pr, order, feat32, cfg.width, cfg.height)
    num_o, den_o = fo.fuse(pr, order, gt, cfg.width, cfg.height)
    touch = pu.Borderline(scene.n, cfg.feat_dim)
    touch.add_view(pr, np.nonzero(o["fragile"])[0], cfg.width, bo, gt)

    gp = pu.GpuPath(scene, cfg.width, cfg.height, 16, surfel=surfel)
    dev = gp.g.mean.device
    W, H, D, n = cfg.width, cfg.height, cfg.feat_dim, scene.n
    vs, bufs = guarded_view_state(fb, torch, n, W, H, bo["M"] + 3, dev, surfel=surfel)   # capacity barely above M: a tail overrun hits the guard
    gp.vs = vs
    es = scene.feat.dtype.itemsize
    outs = dict(rgb=Guarded(torch, 12 * W * H, dev), feat=Guarded(torch, es * W * H * D, dev), T=Guarded(torch, 4 * W * H, dev),
                n=Guarded(torch, 4 * W * H, dev), num=Guarded(torch, 4 * n * D, dev), den=Guarded(torch, 4 * n, dev),
                fused=Guarded(torch, es * n * D, dev), lgt=Guarded(torch, 4 * W * H, dev), lcf=Guarded(torch, 4 * W * H, dev),
                gop=Guarded(torch, 4 * n, dev))
    fdt = torch.float16 if es == 2 else torch.float32
    t_rgb, t_feat = outs["rgb"].view(torch.float32, (H, W, 3)), outs["feat"].view(fdt, (H, W, D))
    t_T, t_n = outs["T"].view(torch.float32, (H, W)), outs["n"].view(torch.int32, (H, W))
    t_num, t_den = outs["num"].view(torch.float32, (n, D)), outs["den"].view(torch.float32, (n,))
    t_fused = outs["fused"].view(fdt, (n, D))
    gt_d = torch.from_numpy(np.ascontiguousarray(gt)).to(dev)
    c = gp.camera(cam)
    first = None
    for rep in range(3):
        for fl in sort_flags:
            for b in bufs.values():
                b.poison(0xFF if rep != 1 else 0x7B)
            fb.project(gp.ctx, gp.g, c, gp.prm, vs)
            m = fb.bin_sort(gp.ctx, c, vs, sync=True, flags=fl)
            pu.check_projection(pr, vs.projected())
            pu.check_bins(bo, vs, m)
        for k in ("rgb", "feat", "T", "n", "num", "den"):
            outs[k].poison()
        fb.render(gp.ctx, gp.g, c, gp.prm, vs, t_rgb, t_feat, t_T, t_n)
        fb.fuse_features(gp.ctx, c, gp.prm, vs, gt_d, t_num, t_den, None, fb.FHGS_FUSE_ZERO)
        t_fused.copy_(torch.from_numpy(scene.feat).to(dev))
        fb.fuse_features(gp.ctx, None, gp.prm, vs, None, t_num, t_den, t_fused, fb.FHGS_FUSE_FINALIZE_ONLY)
        torch.cuda.synchronize()
        g = dict(rgb=t_rgb.cpu().numpy(), feat=t_feat.cpu().numpy(), T=t_T.cpu().numpy(), n=t_n.cpu().numpy())
        assert np.isfinite(g["feat"].astype(np.float32)).all() and np.isfinite(g["rgb"]).all()   # every element written
        pu.check_render(o, g, float(np.abs(feat32).max()), tol)
        pu.check_fuse(num_o, den_o, t_num, t_den, float(np.abs(gt.astype(np.float32)).max()), tol, touch)
        if first is None:
            first = g
        else:
            for k in ("rgb", "feat", "T", "n"):
                assert np.array_equal(first[k], g[k]), f"{k} not reproducible (repetition {rep})"
        if D % 64 != 0:
            # the single-traversal call (per-pixel regime) on poisoned outputs and cleared accumulators: against the oracle
            # directly, and bit for bit against the two separate calls
            for k in ("rgb", "feat", "T", "n"):
                outs[k].poison()
            outs["num"].zero(); outs["den"].zero()
            fb.render_fuse(gp.ctx, gp.g, c, gp.prm, vs, t_rgb, t_feat, gt_d, t_num, t_den, out_T=t_T, out_ncontrib=t_n)
            torch.cuda.synchronize()
            g2 = dict(rgb=t_rgb.cpu().numpy(), feat=t_feat.cpu().numpy(), T=t_T.cpu().numpy(), n=t_n.cpu().numpy())
            for k in g2:
                assert np.array_equal(g[k], g2[k]), f"fhgs_render_fuse: {k} differs from fhgs_render"
            pu.check_fuse(num_o, den_o, t_num, t_den, float(np.abs(gt.astype(np.float32)).max()), tol, touch)
        if ndfd:
            t_lgt, t_lcf = outs["lgt"].view(torch.float32, (H, W)), outs["lcf"].view(torch.float32, (H, W))
            outs["lgt"].poison(); outs["lcf"].poison(); outs["gop"].zero()
            fb.ndfd_forward(gp.ctx, gp.g, c, gp.prm, vs, gt_d, t_lgt, t_lcf)
            work = fb.ndfd_backward(gp.ctx, gp.g, c, gp.prm, vs, gt_d, outs["gop"].view(torch.float32, (n,)))
            torch.cuda.synchronize()
            del work
            assert np.isfinite(t_lgt.cpu().numpy()).all() and np.isfinite(t_lcf.cpu().numpy()).all()
    bad = [k for k, b in list(bufs.items()) + list(outs.items()) if not b.intact()]
    assert not bad, f"guard band overwritten next to: {bad}"
    return dict(M=int(bo["M"]))


def test_guards_pixel_kernels():
    """D = 8 and D = 24 per-pixel kernels, RGB paths, both sort schedules, ragged image."""
    print(run_guarded(inputs.CONFIGS["tiny"], 1, pu.TOL_F32))
    print(run_guarded(pu.reduced_config("tiny", n=3000, feat_dim=24, width=83, height=45), 0, pu.TOL_F32))


def test_guards_ws_kernels_f32():
    """render_ws<128,float> / fuse_ws<float> (D = 128, 256), render_ws<64> / fuse_tiled<64> (D = 64, 192), ragged tiles,
    plus the NDFD forward / backward kernels on the same view state."""
    print(run_guarded(pu.reduced_config("mid", n=20_000, width=200, height=120, log_scale_mu=-3.2), 0, pu.TOL_F32, ndfd=True))
    print(run_guarded(pu.reduced_config("mid", n=8_000, width=120, height=72, log_scale_mu=-3.0, feat_dim=256), 0, pu.TOL_F32,
                      sort_flags=(0,), ndfd=True))
    for d in (64, 192):
        print(run_guarded(pu.reduced_config("mid", n=8_000, width=120, height=72, log_scale_mu=-3.0, feat_dim=d), 0, pu.TOL_F32,
                          sort_flags=(0,), ndfd=(d == 64)))


def test_guards_ws_kernels_f16():
    """render_ws<128,__half> / fuse_ws<__half> at D = 512 (four channel chunks) and D = 128."""
    print(run_guarded(pu.reduced_config("large", n=12_000, width=136, height=88, log_scale_mu=-3.2), 0, pu.TOL_F16, sort_flags=(0,)))
    print(run_guarded(pu.reduced_config("large", n=12_000, width=136, height=88, log_scale_mu=-3.2, feat_dim=128), 0, pu.TOL_F16,
                      sort_flags=(0,)))


def test_guards_surfel_kernels():
    """FHGS_PRIM_SURFEL: project_surfel_kernel, the surfel forms of render_ws<128> / fuse_ws (288-slot ring), render_ws<64> /
    fuse_tiled<64>, the per-pixel kernels (D = 24), fp16 storage, and the surfel NDFD forward, between guard bands, on
    poisoned buffers (ray_transform included), three times."""
    print(run_guarded(pu.reduced_config("mid", n=20_000, width=200, height=120, log_scale_mu=-2.8), 0, pu.TOL_F32, ndfd=True, surfel=True))
    print(run_guarded(pu.reduced_config("mid", n=8_000, width=120, height=72, log_scale_mu=-2.6, feat_dim=64), 0, pu.TOL_F32,
                      sort_flags=(0,), surfel=True))
    print(run_guarded(pu.reduced_config("tiny", n=3000, feat_dim=24, width=83, height=45, log_scale_mu=-2.3), 0, pu.TOL_F32, surfel=True))
    print(run_guarded(pu.reduced_config("large", n=12_000, width=136, height=88, log_scale_mu=-2.8, feat_dim=128), 0, pu.TOL_F16,
                      sort_flags=(0,), surfel=True))


def test_fuse_ws_back_to_back_stress():
    """The fuse pipeline hands partial sums between its pixel halves through mbarriers and, for an fp32 map with D > 128,
    consumes the GT tile while it streams in: 60 back-to-back accumulations of the same view without a host sync (D = 128
    and D = 256, fp32) must complete (an mbarrier over-arrival traps) and reproduce the first one up to the atomic order."""
    import torch
    from paper_2505_19154_b200 import binding as fb
    for d in (128, 256):
        cfg = pu.reduced_config("multiview", n=60_000, width=432, height=328, n_views=200, log_scale_mu=-3.0, feat_dim=d)
        scene = inputs.make_scene(cfg)
        cam = inputs.make_camera(cfg, 25)
        gp = pu.GpuPath(scene, cfg.width, cfg.height, 12_000_000)
        c, m = gp.project_sort(cam)
        dev = gp.g.mean.device
        gt = torch.from_numpy(inputs.make_gt_map(cfg, 25, cam)).to(dev)
        num = torch.zeros((scene.n, d), dtype=torch.float32, device=dev)
        den = torch.zeros((scene.n,), dtype=torch.float32, device=dev)
        fb.fuse_features(gp.ctx, c, gp.prm, gp.vs, gt, num, den, None, fb.FHGS_FUSE_ZERO)
        torch.cuda.synchronize()
        num0, den0 = num.clone(), den.clone()
        assert float(den0.sum()) > 1000.0
        reps = 60
        for _ in range(reps):
            fb.project(gp.ctx, gp.g, c, gp.prm, gp.vs)
            fb.bin_sort(gp.ctx, c, gp.vs, sync=False)
            fb.fuse_features(gp.ctx, c, gp.prm, gp.vs, gt, num, den, None, 0)
        torch.cuda.synchronize()
        k = reps + 1
        assert float((den - k * den0).abs().max()) <= 2e-5 * k * float(den0.max())
        assert float((num - k * num0).abs().max()) <= 2e-5 * k * float(num0.abs().max())

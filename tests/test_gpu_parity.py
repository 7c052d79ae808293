"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Bars (north_star / SURVEY 8(c)): integers bit-exact (radius, rect,
tiles_touched, M, offsets, sorted keys AND values, ranges, n_contrib off fragile pixels); fp32
RGB / features / T / fused vectors within 1e-4 max abs; 2e-3 where features are stored fp16."""
import numpy as np
import pytest

from oracle import fhgs_oracle as fo
from paper_2505_19154_b200 import inputs
import parity_util as pu

pytestmark = pytest.mark.gpu


def run_case(cfg, views, tol, literal_pixels=None, sort_flags=(0, 1), capacity_slack=1.25, check_finalize=True,
             fixed_capacity=None, full_frame=True, rect_mode=0, primitive=0):
    """Full P -> S -> R -> F parity of one config over `views`; returns worst errors.
    full_frame: compare the whole rendered frame with fo_render_scatter; literal_pixels: additionally (or instead)
    compare that many random pixels with the tile-free, box-free fo_render_literal.  Fusion is always compared on
    every row of num / den and on every finalised vector."""
    import time
    scene = inputs.make_scene(cfg)
    cams = [inputs.make_camera(cfg, v) for v in views]
    prm_o = fo.params(rect_mode=rect_mode, primitive=primitive)
    prs = [pu.oracle_view(scene, cam, prm_o) for cam in cams]
    Ms = [int(pr["tiles_touched"].astype(np.int64).sum()) for pr in prs]
    cap = int(max(Ms) * capacity_slack) + 16
    if fixed_capacity is not None:
        cap = fixed_capacity
    gp = pu.GpuPath(scene, cfg.width, cfg.height, cap, surfel=bool(primitive), storage=cfg.feat_dtype)
    gp.prm.rect_mode = rect_mode
    feat32 = scene.feat.astype(np.float32)
    fabs = float(np.abs(feat32).max())
    worst = {"M": max(Ms)}
    num_o = np.zeros((scene.n, cfg.feat_dim)); den_o = np.zeros(scene.n)
    num_g = den_g = None
    border = pu.Borderline(scene.n, cfg.feat_dim)
    t_oracle = 0.0
    for vi, (v, cam, pr) in enumerate(zip(views, cams, prs)):
        t0 = time.time()
        bo = fo.bins(pr, cfg.width, cfg.height)
        t_oracle += time.time() - t0
        for fl in sort_flags:
            c, m = gp.project_sort(cam, flags=fl)
            pu.check_projection(pr, gp.vs.projected())
            pu.check_bins(bo, gp.vs, m)
        order = fo.global_order(pr)
        g = gp.render(c)
        fpix = None
        if full_frame:
            t0 = time.time()
            o = fo.render_scatter(pr, order, feat32, cfg.width, cfg.height)
            t_oracle += time.time() - t0
            w = pu.check_render(o, g, fabs, tol)
            fpix = np.nonzero(o["fragile"])[0]
            del o
            for k, val in w.items():
                worst[k] = max(worst.get(k, 0), val)
        if literal_pixels is not None:
            rng = np.random.default_rng(7 + v)
            pix = np.unique(rng.integers(0, cfg.width * cfg.height, size=literal_pixels)).astype(np.int32)
            o = fo.render_literal(pr, order, feat32, cfg.width, cfg.height, pix=pix)
            w = pu.check_render(o, g, fabs, tol, pix=pix)
            for k, val in w.items():
                worst["lit_" + k] = max(worst.get("lit_" + k, 0), val)
        if fpix is None:   # fragile pixels of the whole frame (RGB-only scatter pass: no feature work)
            fpix = np.nonzero(fo.render_scatter(pr, order, None, cfg.width, cfg.height)["fragile"])[0]
        del g
        # fusion, accumulated over the views
        gt = inputs.make_gt_map(cfg, v, cam)
        gabs = float(np.abs(gt.astype(np.float32)).max())
        t0 = time.time()
        fo.fuse(pr, order, gt, cfg.width, cfg.height, num=num_o, den=den_o)
        t_oracle += time.time() - t0
        border.add_view(pr, fpix, cfg.width, bo, gt)
        del bo
        fl = None if vi == 0 else 0
        num_g, den_g = gp.fuse(c, gt, num_g, den_g, flags=fl)
        del gt
    w = pu.check_fuse(num_o, den_o, num_g, den_g, gabs, tol, border)
    worst.update({"fuse_" + k: val for k, val in w.items()})
    if check_finalize:
        f_o = fo.finalize(num_o, den_o, feat32)
        f_g = gp.finalize(num_g, den_g, scene.feat)
        den_gn = den_g.cpu().numpy()
        worst["fused"], worst["fused_rows"], worst["fused_rows_alt"], _ = pu.check_finalized(
            f_o, f_g, scene.feat, num_o, den_o, den_gn, tol, border=border)
        # rows nobody blends keep their previous value exactly
        keep = (den_o == 0) & (den_gn == 0)
        assert np.array_equal(f_g[keep], scene.feat[keep])
    worst["borderline_fragments"] = len(border.g)
    worst["oracle_s"] = round(t_oracle, 1)
    return worst


def test_tiny_all_views():
    """configs[0]: N=1000, D=8, 64x64, 4 views (per-pixel kernels, CH=8)."""
    w = run_case(inputs.CONFIGS["tiny"], range(4), pu.TOL_F32)
    print(w)


def test_small_full():
    """configs[1] as BASELINE.json states it: N=10^5, SH degree 1, D=16, all 8 views at 256x256 fused into one
    accumulator, both sort schedules; every frame compared whole, plus 200 pixels per view with the literal oracle."""
    w = run_case(inputs.CONFIGS["small"], range(8), pu.TOL_F32, literal_pixels=200)
    print(w)


def test_mid_shape_ragged_tiles_d128():
    """configs[2] shape at reduced size: D=128 unit features (tiled kernels, DC=128), SH degree 3,
    328x200 px: 20.5 x 12.5 tiles -> ragged right column and bottom row."""
    cfg = pu.reduced_config("mid", n=60_000, width=328, height=200, log_scale_mu=-3.3)
    w = run_case(cfg, [0], pu.TOL_F32)
    print(w)


def test_d64_and_d192_paths():
    """DC=64 kernels: D=64 (one pass) and D=192 (three passes)."""
    for d in (64, 192):
        cfg = pu.reduced_config("mid", n=15_000, width=160, height=96, log_scale_mu=-3.0, feat_dim=d)
        print(d, run_case(cfg, [0], pu.TOL_F32, sort_flags=(0,)))


def test_multiview_shape_d256():
    """configs[4] shape at reduced size: blobs, D=256 (two channel passes), 3 orbit views accumulated."""
    cfg = pu.reduced_config("multiview", n=40_000, width=216, height=168, n_views=200, log_scale_mu=-3.0)
    w = run_case(cfg, [0, 67, 133], pu.TOL_F32, sort_flags=(0,))
    print(w)


def test_large_shape_fp16_d512():
    """configs[3] shape at reduced size: D=512 stored fp16, accumulated fp32, fp16 image / fused output."""
    cfg = pu.reduced_config("large", n=30_000, width=200, height=120, log_scale_mu=-3.3)
    w = run_case(cfg, [0], pu.TOL_F16, sort_flags=(0,))
    print(w)


def test_fp16_storage_d256_multiview_shape():
    """fp16 storage at D = 256 (features, GT map, feature image and fused output in fp16, fp32
    accumulation) on the Multi-view shape: blobs, 3 orbit views accumulated, 2e-3."""
    cfg = pu.reduced_config("multiview", n=40_000, width=216, height=168, n_views=200, log_scale_mu=-3.0, feat_dtype="f16")
    w = run_case(cfg, [0, 67, 133], pu.TOL_F16, sort_flags=(0,))
    print(w)


def test_bf16_storage_d256_and_d64():
    """NEXT-4 (iv): bfloat16 storage of feature rows, GT maps and feature outputs (fp32 arithmetic), on the warp-specialised
    kernels (D = 256: two channel chunks, double-buffered 16-bit GT tile) and the tiled ones (D = 64)."""
    cfg = pu.reduced_config("multiview", n=40_000, width=216, height=168, n_views=200, log_scale_mu=-3.0, feat_dtype="bf16")
    w = run_case(cfg, views=[0, 100], tol=pu.TOL_BF16)
    print("bf16 d256", w)
    cfg = pu.reduced_config("mid", n=30_000, width=200, height=120, log_scale_mu=-3.0, feat_dim=64, feat_dtype="bf16")
    w = run_case(cfg, views=[0], tol=pu.TOL_BF16)
    print("bf16 d64", w)
    # the NDFD entry points take f32 / f16 only and say so
    import torch
    from paper_2505_19154_b200 import binding as fb
    scene = inputs.make_scene(cfg)
    cam = inputs.make_camera(cfg, 0)
    gp = pu.GpuPath(scene, cfg.width, cfg.height, 1 << 20, storage="bf16")
    c, _ = gp.project_sort(cam)
    gt = torch.zeros((cfg.height, cfg.width, cfg.feat_dim), dtype=torch.bfloat16, device="cuda")
    lgt = torch.zeros((cfg.height, cfg.width), dtype=torch.float32, device="cuda")
    with pytest.raises(fb.FhgsError) as e:
        fb.ndfd_forward(gp.ctx, gp.g, c, gp.prm, gp.vs, gt, lgt, lgt.clone())
    assert e.value.status == fb.FHGS_ERR_INVALID


def test_odd_d_paths():
    """D=4 and D=24 (CH=4 / CH=8 per-pixel kernels)."""
    for d in (4, 24):
        cfg = pu.reduced_config("tiny", n=3000, feat_dim=d, width=80, height=48)
        print(d, run_case(cfg, [1], pu.TOL_F32, sort_flags=(0,)))


def test_mid_full_size_bench_configuration():
    """configs[2] at FULL size, exactly as bench.py launches it (N=10^6, SH3, D=128 fp32, 1920x1080, default sort
    schedule, capacity 40e6): every integer output bit-exact (radius, rect, tiles_touched, M, offsets, all 3.2e7 sorted
    keys and values, ranges, n_contrib), every float of the image / feature image / fused vectors within 1e-4."""
    cfg = inputs.CONFIGS["mid"]
    w = run_case(cfg, [0], pu.TOL_F32, sort_flags=(0,), capacity_slack=1.0, fixed_capacity=int(40e6))
    print(w)


def test_tight_rect_mode():
    """SURVEY 8(f) NEXT-4 (i), fhgs_params.rect_mode = FHGS_RECT_TIGHT: per-axis 3-sigma tile rectangles.  Same parity
    bars (rect, tiles_touched, M, all sorted pairs, ranges bit-exact against the oracle run with the same rule; images
    and fused vectors within 1e-4 of the oracle, whose renderer does not depend on the rule) on the Tiny config, a
    ragged D=128 case and the Mid config at FULL size, where it must shed at least a third of the instances."""
    print(run_case(inputs.CONFIGS["tiny"], range(4), pu.TOL_F32, rect_mode=1))
    cfg = pu.reduced_config("mid", n=60_000, width=328, height=200, log_scale_mu=-3.3)
    print(run_case(cfg, [0], pu.TOL_F32, rect_mode=1))
    w = run_case(inputs.CONFIGS["mid"], [0], pu.TOL_F32, sort_flags=(0,), capacity_slack=1.0, fixed_capacity=int(40e6), rect_mode=1)
    print(w)
    assert w["M"] < 0.67 * 31_666_264


def test_surfel_primitive():
    """SURVEY 8(f) NEXT-3, fhgs_params.primitive = FHGS_PRIM_SURFEL: the paper's 2-D surfel with exact ray-splat
    intersection.  Same bars as the EWA path: ray transform, bounding box, rect, tiles_touched, M, all
    sorted pairs and ranges bit-exact; n_contrib exact off fragile pixels; images, accumulators and fused vectors within
    1e-4 (2e-3 for fp16 storage).  Tiny-shape (4 views, per-pixel kernels), Small-shape (2 views accumulated), a ragged
    D=128 case (16-channel render passes, tile-GEMM fusion), D=64 and fp16 storage."""
    print(run_case(pu.reduced_config("tiny", n=3000, log_scale_mu=-2.3), range(4), pu.TOL_F32, primitive=1, literal_pixels=150))
    print(run_case(pu.reduced_config("small", n=20_000, log_scale_mu=-2.6), [0, 3], pu.TOL_F32, primitive=1, sort_flags=(0,)))
    print(run_case(pu.reduced_config("mid", n=40_000, width=328, height=200, log_scale_mu=-2.8), [0], pu.TOL_F32, primitive=1, sort_flags=(0,)))
    print(run_case(pu.reduced_config("mid", n=10_000, width=160, height=96, log_scale_mu=-2.6, feat_dim=64), [0], pu.TOL_F32, primitive=1, sort_flags=(0,)))
    print(run_case(pu.reduced_config("large", n=15_000, width=200, height=120, log_scale_mu=-2.8), [0], pu.TOL_F16, primitive=1, sort_flags=(0,)))


def test_large_full_size():
    """configs[3] at FULL size (N=3*10^6, D=512 fp16, 1920x1080): projection and the whole sorted instance list
    (9.5e7 pairs) bit-exact; the whole 1080p x 512-channel feature image, T, n_contrib against fo_render_scatter and
    300 random pixels against the literal per-pixel oracle; all 3*10^6 x 512 accumulator rows, den and every
    finalised (fp16) vector against fo_fuse_scatter (fuse_ws_kernel<__half>, 4 channel chunks) at 2e-3."""
    cfg = inputs.CONFIGS["large"]
    w = run_case(cfg, [0], pu.TOL_F16, literal_pixels=300, sort_flags=(0,), capacity_slack=1.02)
    print(w)


def test_multiview_full_size_eight_views():
    """configs[4] at FULL size (N=2*10^6 in 64 blobs, D=256 fp32, 1296x968), views {0,25,...,175} of the 200-camera
    orbit fused into one accumulator: full element-by-element parity of P, S, R, F."""
    cfg = inputs.CONFIGS["multiview"]
    w = run_case(cfg, range(0, 200, 25), pu.TOL_F32, sort_flags=(0,), capacity_slack=1.02)
    print(w)


def test_randomized_shapes_sweep():
    """16 seeded random cases: scene family, N, odd image sizes (ragged tiles in both directions, images narrower than
    a tile row), D over every kernel variant (4..512, fp32/fp16), splat size, camera; full P/S/R/F parity each."""
    rng = np.random.default_rng(20251104)
    for it in range(16):
        base = str(rng.choice(["tiny", "mid", "multiview", "large"]))
        d = int(rng.choice([4, 8, 16, 24, 64, 128, 192, 256] if base != "large" else [64, 128, 256, 512]))
        kw = dict(n=int(rng.integers(200, 25000)), width=int(rng.integers(17, 400)), height=int(rng.integers(17, 300)),
                  feat_dim=d, log_scale_mu=float(rng.uniform(-4.0, -2.0)), seed=int(rng.integers(1, 10 ** 6)))
        if base == "multiview":
            kw["n_views"] = 200
        cfg = pu.reduced_config(base, **kw)
        view = int(rng.integers(0, cfg.n_views))
        w = run_case(cfg, [view], pu.TOL_F16 if base == "large" else pu.TOL_F32, sort_flags=(0, 1) if it % 4 == 0 else (0,))
        print(it, base, kw, view, w)


def test_project_sh_row_paths_agree():
    """Step P at SH degree 3 has two ways to fetch a Gaussian's SH row: one bulk async copy per row (16-byte aligned sh
    array) and the CTA-staged form (any alignment).  Both must give the oracle's projection, bit for bit on everything but
    the colour, and the same colour bits as each other -- also when most of the frame test's guesses are wrong (a camera
    that sees only part of the scene, so many staged rows belong to Gaussians that are culled later and vice versa)."""
    import torch
    from paper_2505_19154_b200 import binding as fb
    cfg = inputs.scaled(inputs.CONFIGS["mid"], n=70001, width=208, height=112, log_scale_mu=-2.5, n_views=4)
    scene = inputs.make_scene(cfg)
    assert scene.sh_degree == 3
    ctx = fb.Context(0)
    prm = fb.default_params()
    g = fb.Gaussians(scene.mean, scene.scale, scene.quat, scene.opacity, scene.sh, None, scene.sh_degree)
    # the same coefficients at an address that is 4 (mod 16): the staged form
    raw = torch.empty(g.sh.numel() + 4, dtype=torch.float32, device="cuda")
    base = 1 if raw.data_ptr() % 16 == 0 else 0
    while (raw.data_ptr() + 4 * base) % 16 == 0:
        base += 1
    sh_off = raw[base:base + g.sh.numel()].view_as(g.sh)
    sh_off.copy_(g.sh)
    g2 = fb.Gaussians(scene.mean, scene.scale, scene.quat, scene.opacity, scene.sh, None, scene.sh_degree)
    g2.sh = sh_off
    g2.refresh()
    assert g.sh.data_ptr() % 16 == 0 and g2.sh.data_ptr() % 16 != 0
    for view in (0, 1):
        cam = inputs.make_camera(cfg, view)
        c = fb.make_camera(cam.view, cam.proj, cam.cam_pos, cam.width, cam.height)
        pr = pu.oracle_view(scene, cam)
        outs = []
        for gg in (g, g2):
            vs = fb.ViewState(scene.n, cfg.width, cfg.height, 0)
            vs.rgb.fill_(float("nan"))
            fb.project(ctx, gg, c, prm, vs)
            torch.cuda.synchronize()
            outs.append(vs.projected())
            pu.check_projection(pr, outs[-1])
        for k in outs[0]:
            assert np.array_equal(outs[0][k].view(np.uint8), outs[1][k].view(np.uint8)), f"paths differ in {k} (view {view})"
        assert 0 < int((outs[0]["tiles_touched"] > 0).sum()) < scene.n


@pytest.mark.parametrize("case", ["tiny", "small", "d48_f16", "surfel_d24"])
def test_render_fuse_single_traversal(case):
    """NEXT-4 (ii): fhgs_render_fuse (one traversal, one weight phase) against fhgs_render followed by fhgs_fuse_features on
    the same view state: images and contributor counts bit for bit, accumulators (two views accumulated) up to the order
    of their floating-point atomics; the separate calls are the ones the oracle checks element by element above."""
    import torch
    from paper_2505_19154_b200 import binding as fb
    surfel = case == "surfel_d24"
    if case == "tiny":
        cfg = inputs.CONFIGS["tiny"]
    elif case == "small":
        cfg = inputs.CONFIGS["small"]
    elif case == "d48_f16":
        cfg = pu.reduced_config("small", n=30_000, width=200, height=120, feat_dim=48, feat_dtype="f16")
    else:
        cfg = pu.reduced_config("small", n=20_000, width=136, height=88, feat_dim=24)
    scene = inputs.make_scene(cfg)
    W, H, D, n = cfg.width, cfg.height, cfg.feat_dim, scene.n
    gp = pu.GpuPath(scene, W, H, 64 * n + 4096, surfel=surfel)
    dev = gp.g.mean.device
    fdt = gp.g.feat.dtype
    mk = lambda: dict(rgb=torch.full((H, W, 3), float("nan"), device=dev), feat=torch.zeros((H, W, D), dtype=fdt, device=dev),
                      T=torch.full((H, W), float("nan"), device=dev), n=torch.full((H, W), -1, dtype=torch.int32, device=dev))
    num_a, den_a = torch.zeros((n, D), device=dev), torch.zeros((n,), device=dev)
    num_b, den_b = torch.zeros((n, D), device=dev), torch.zeros((n,), device=dev)
    gmax = 0.0
    for view in (0, 1):
        cam = inputs.make_camera(cfg, view)
        c, m = gp.project_sort(cam)
        assert m > 0
        gt = torch.from_numpy(np.ascontiguousarray(inputs.make_gt_map(cfg, view, cam))).to(dev)
        gmax = max(gmax, float(gt.float().abs().max()))
        a, b = mk(), mk()
        fb.render(gp.ctx, gp.g, c, gp.prm, gp.vs, a["rgb"], a["feat"], a["T"], a["n"])
        fb.fuse_features(gp.ctx, c, gp.prm, gp.vs, gt, num_a, den_a, None, 0)
        fb.render_fuse(gp.ctx, gp.g, c, gp.prm, gp.vs, b["rgb"], b["feat"], gt, num_b, den_b, out_T=b["T"], out_ncontrib=b["n"])
        torch.cuda.synchronize()
        for k in a:
            assert torch.equal(a[k], b[k]), f"{k} differs (view {view})"
    assert bool((den_a > 0).any())
    assert bool(((den_a - den_b).abs() <= pu.TOL_F32 * den_a.abs() + 1e-12).all())
    assert bool(((num_a - num_b).abs().amax(dim=1) <= pu.TOL_F32 * den_a.abs() * gmax + 1e-12).all())
    # the tiled regime is refused with a message that says why
    if case == "tiny":
        cfg64 = pu.reduced_config("tiny", feat_dim=64)
        sc64 = inputs.make_scene(cfg64)
        gp64 = pu.GpuPath(sc64, cfg64.width, cfg64.height, 1 << 16)
        c64, _ = gp64.project_sort(inputs.make_camera(cfg64, 0))
        z = lambda *s: torch.zeros(s, device=dev)
        with pytest.raises(fb.FhgsError) as e:
            fb.render_fuse(gp64.ctx, gp64.g, c64, gp64.prm, gp64.vs, z(64, 64, 3), z(64, 64, 64), z(64, 64, 64), z(sc64.n, 64), z(sc64.n))
        assert e.value.status == fb.FHGS_ERR_INVALID and "multiple of 64" in str(e.value)


def test_large_tile_grid_fallback_sort():
    """2064x1616 px -> (GW+1)*(GH+1) = 130*102 > 12288: fhgs_bin_sort leaves the shared-memory tile-count
    path and derives histograms / ranges from the instance list; both schedules, integers bit-exact."""
    cfg = pu.reduced_config("tiny", n=4000, width=2064, height=1616, log_scale_mu=-2.2)
    scene = inputs.make_scene(cfg)
    cam = inputs.make_camera(cfg, 1)
    pr = pu.oracle_view(scene, cam)
    bo = fo.bins(pr, cfg.width, cfg.height)
    gp = pu.GpuPath(scene, cfg.width, cfg.height, bo["M"] + 7)
    for fl in (0, 1):
        c, m = gp.project_sort(cam, flags=fl)
        pu.check_projection(pr, gp.vs.projected())
        pu.check_bins(bo, gp.vs, m)
    print("M =", bo["M"])


def test_edge_cases():
    import torch
    from paper_2505_19154_b200 import binding as fb
    cfg = inputs.CONFIGS["tiny"]
    scene = inputs.make_scene(cfg)
    cam = inputs.make_camera(cfg, 0)
    # (a) nothing visible: every Gaussian behind the camera -> M = 0, background image, num/den untouched
    behind = inputs.Scene(scene.mean + np.array([0, 0, -100], np.float32), scene.scale, scene.quat, scene.opacity,
                          scene.sh, scene.feat, scene.sh_degree)
    gp = pu.GpuPath(behind, 64, 64, 1024)
    gp.prm = fb.default_params(bg=(0.25, 0.5, 0.75))
    c, m = gp.project_sort(cam)
    assert m == 0 and int(gp.vs.ranges.abs().sum()) == 0
    g = gp.render(c)
    assert np.all(g["n"] == 0) and np.all(g["T"] == 1.0) and np.all(g["feat"] == 0)
    assert np.allclose(g["rgb"], np.array([0.25, 0.5, 0.75], np.float32))
    num, den = gp.fuse(c, inputs.make_gt_map(cfg, 0))
    assert float(num.abs().sum()) == 0 and float(den.abs().sum()) == 0
    # (b) capacity overflow: synchronous bin_sort reports it, M is still exact, ranges stay empty
    pr = pu.oracle_view(scene, cam)
    m_true = fo.bins(pr, 64, 64)["M"]
    gp2 = pu.GpuPath(scene, 64, 64, m_true - 1)
    cc = gp2.camera(cam)
    fb.project(gp2.ctx, gp2.g, cc, gp2.prm, gp2.vs)
    with pytest.raises(fb.FhgsError) as ei:
        fb.bin_sort(gp2.ctx, cc, gp2.vs, sync=True)
    assert ei.value.status == fb.FHGS_ERR_CAPACITY
    assert int(gp2.vs.num_instances.item()) == m_true and int(gp2.vs.ranges.abs().sum()) == 0
    # exactly enough capacity works
    gp3 = pu.GpuPath(scene, 64, 64, m_true)
    c3, m3 = gp3.project_sort(cam)
    assert m3 == m_true
    # (c) invalid arguments are rejected before anything is enqueued
    bad = fb.make_camera(cam.view, cam.proj, cam.cam_pos, 0, 64)
    with pytest.raises(fb.FhgsError) as ei:
        fb.project(gp3.ctx, gp3.g, bad, gp3.prm, gp3.vs)
    assert ei.value.status == fb.FHGS_ERR_INVALID
    with pytest.raises(fb.FhgsError):
        fb.render(gp3.ctx, gp3.g, c3, gp3.prm, gp3.vs, None)
    # (d) n = 0
    empty = inputs.Scene(scene.mean[:0], scene.scale[:0], scene.quat[:0], scene.opacity[:0], scene.sh[:0],
                         scene.feat[:0], scene.sh_degree)
    gp4 = pu.GpuPath(empty, 64, 64, 16)
    c4, m4 = gp4.project_sort(cam)
    assert m4 == 0
    # (e) RGB-only render (no features) equals the RGB of the feature render
    g_full = gp3.render(c3)
    g_rgb = gp3.render(c3, with_feat=False)
    assert np.array_equal(g_full["rgb"], g_rgb["rgb"]) and np.array_equal(g_full["n"], g_rgb["n"])
    # (f) determinism of P, S, R
    g_again = gp3.render(c3)
    for k in ("rgb", "feat", "T", "n"):
        assert np.array_equal(g_full[k], g_again[k])


def test_frame_host_equals_stepwise_calls():
    """fhgs_frame_host (HOST buffers, copies overlapped with the steps on the context's copy streams) returns exactly
    what the four calls return when issued one by one (P, S, R are deterministic; fused vectors up to atomic order).
    Run twice with different host data to catch a copy racing a kernel of the previous frame."""
    import torch
    from paper_2505_19154_b200 import binding as fb
    cfg = pu.reduced_config("mid", n=50_000, width=328, height=200, log_scale_mu=-3.3)
    for seed_shift in (0, 1):
        cfg_i = inputs.scaled(cfg, seed=cfg.seed + seed_shift)
        scene = inputs.make_scene(cfg_i)
        cam = inputs.make_camera(cfg_i, 0)
        gt = inputs.make_gt_map(cfg_i, 0, cam)
        if seed_shift == 0:
            gp = pu.GpuPath(scene, cfg.width, cfg.height, 3_000_000)
            dev = gp.g.mean.device
        W, H, D, n = cfg.width, cfg.height, cfg.feat_dim, scene.n
        c = gp.camera(cam)
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        host = dict(mean=pin(scene.mean), scale=pin(scene.scale), quat=pin(scene.quat), opacity=pin(scene.opacity),
                    sh=pin(scene.sh), feat=pin(scene.feat), gt=pin(gt),
                    out_rgb=torch.zeros((H, W, 3)).pin_memory(), out_feat=torch.zeros((H, W, D)).pin_memory(),
                    fused_feat=torch.zeros((n, D)).pin_memory())
        f32 = torch.float32
        ws = dict(out_rgb=torch.empty((H, W, 3), dtype=f32, device=dev), out_feat=torch.empty((H, W, D), dtype=f32, device=dev),
                  gt=torch.empty((H, W, D), dtype=f32, device=dev), num=torch.empty((n, D), dtype=f32, device=dev),
                  den=torch.empty((n,), dtype=f32, device=dev), fused_feat=torch.from_numpy(scene.feat).to(dev))
        m = fb.frame_host(gp.ctx, host, gp.g, c, gp.prm, gp.vs, ws)
        # the same frame, step by step, from the device copies frame_host left in gp.g
        c2, m2 = gp.project_sort(cam)
        assert m == m2
        g = gp.render(c2)
        num, den = gp.fuse(c2, gt)
        fused = gp.finalize(num, den, scene.feat)
        assert np.array_equal(host["out_rgb"].numpy(), g["rgb"])
        assert np.array_equal(host["out_feat"].numpy(), g["feat"])
        # every finalised row (den > den_eps; both runs are the GPU path, they differ by the atomic order only --
        # a relative 1e-6 on num and den -- so rows within 1e-5 of den_eps may be finalised in one run only)
        dn = den.cpu().numpy().astype(np.float64)
        seen = dn > 1e-8 * (1 + 1e-5)
        assert seen.sum() > 1000
        assert np.abs(host["fused_feat"].numpy()[seen] - fused[seen]).max() <= 1e-5
        never = dn == 0
        assert np.array_equal(host["fused_feat"].numpy()[never], scene.feat[never])


def test_tile_visited_diagnostics():
    """fhgs_render's per-tile 'visited' diagnostics (work accounting only): never longer than the tile's list; the
    Tiny scene never saturates, so every tile walks its whole list; a saturating scene stops early somewhere."""
    for name, kw, saturates in (("tiny", {}, False), ("mid", dict(n=60_000, width=328, height=200, log_scale_mu=-3.3), True)):
        cfg = pu.reduced_config(name, **kw) if kw else inputs.CONFIGS[name]
        scene = inputs.make_scene(cfg)
        cam = inputs.make_camera(cfg, 0)
        gp = pu.GpuPath(scene, cfg.width, cfg.height, 4_000_000)
        c, m = gp.project_sort(cam)
        gp.ctx.set_diagnostics(True)
        g_diag = gp.render(c)
        gp.ctx.set_diagnostics(False)
        g_plain = gp.render(c)
        for k in ("rgb", "feat", "T", "n"):
            assert np.array_equal(g_diag[k], g_plain[k])   # the diagnostics variant computes the same image
        tv = gp.vs.tile_visited().cpu().numpy().astype(np.int64)
        rg = gp.vs.ranges.cpu().numpy().view(np.uint32).astype(np.int64)
        ln = rg[:, 1] - rg[:, 0]
        assert np.all(tv <= ln) and np.all(tv[ln > 0] > 0)
        if saturates:
            assert np.any(tv < ln)
        else:
            assert np.array_equal(tv, ln)


def test_constant_map_and_l2norm():
    """north_star pin on the GPU path: a constant GT map fuses to that constant; L2NORM normalises."""
    cfg = inputs.CONFIGS["tiny"]
    scene = inputs.make_scene(cfg)
    cam = inputs.make_camera(cfg, 2)
    gp = pu.GpuPath(scene, 64, 64, 8192)
    c, m = gp.project_sort(cam)
    v = np.linspace(-2.0, 3.0, cfg.feat_dim).astype(np.float32)
    gt = np.broadcast_to(v, (64, 64, cfg.feat_dim)).copy()
    num, den = gp.fuse(c, gt)
    f = gp.finalize(num, den, scene.feat)
    seen = den.cpu().numpy() > 1e-6
    assert seen.sum() > 100
    assert np.abs(f[seen] - v).max() <= 1e-4
    fn = gp.finalize(num, den, scene.feat, l2norm=True)
    assert np.abs(fn[seen] - v / np.linalg.norm(v)).max() <= 1e-4


def test_zero_touched_equals_full_clear():
    """FHGS_FUSE_ZERO_TOUCHED clears exactly what a full clear clears when the buffers were maintained by the library:
    after it num and den are all zero, and a second accumulation reproduces the first (up to the atomic order)."""
    import torch
    from paper_2505_19154_b200 import binding as fb
    cfg = pu.reduced_config("mid", n=30_000, width=200, height=120, log_scale_mu=-3.2)
    scene = inputs.make_scene(cfg)
    cam = inputs.make_camera(cfg, 0)
    gt = inputs.make_gt_map(cfg, 0, cam)
    gp = pu.GpuPath(scene, cfg.width, cfg.height, 3_000_000)
    c, m = gp.project_sort(cam)
    num, den = gp.fuse(c, gt)                                      # full clear + accumulate
    num1, den1 = num.clone(), den.clone()
    assert int((den1 != 0).sum()) > 1000
    fb.fuse_features(gp.ctx, None, gp.prm, gp.vs, None, num, den, None, fb.FHGS_FUSE_ZERO_ONLY | fb.FHGS_FUSE_ZERO_TOUCHED)
    torch.cuda.synchronize()
    assert float(num.abs().max()) == 0.0 and float(den.abs().max()) == 0.0
    num, den = gp.fuse(c, gt, num, den, flags=fb.FHGS_FUSE_ZERO | fb.FHGS_FUSE_ZERO_TOUCHED)
    assert torch.equal(den != 0, den1 != 0)
    assert float((den - den1).abs().max()) <= 1e-5 * float(den1.abs().max())
    assert float((num - num1).abs().max()) <= 1e-5 * float(num1.abs().max())
    with pytest.raises(fb.FhgsError):                               # ZERO_TOUCHED alone means nothing
        fb.fuse_features(gp.ctx, c, gp.prm, gp.vs, torch.from_numpy(gt).to(num.device), num, den, None, fb.FHGS_FUSE_ZERO_TOUCHED)


def test_multiview_sweep_driver_small():
    """bench.py's 200-view sweep driver (BASELINE.json configs[4]; parallel.fuse_views_sharded with the CUDA calls, maps
    generated on the device) at debug size, 12 views, one rank: runs, conserves weight, and the fused vectors of
    well-covered Gaussians point at their blob's vector."""
    import json, os, subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--workload", "multiview", "--views", "12", "--small"],
                       capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    inv = line["invariants"]
    print(line["ms"], inv)
    assert inv["conservation_rel_err"] < 2e-4
    assert inv["cosine_to_blob_vector"]["gaussians"] > 1000 and inv["cosine_to_blob_vector"]["median"] > 0.9

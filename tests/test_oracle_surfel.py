"""Pins for the surfel variant of the CPU oracle (Eq. 1-3): SPEC.md's worked
intersection values, reprojection consistency against an independent pinhole written here in numpy/float64, the
conservative screen bounds by exhaustive scan, culling cases, the small-splat limit in which the surfel and the EWA
Gaussian agree, literal == scatter, and the compositing / fusion invariants in surfel mode.  CPU only."""
import math

import numpy as np
import pytest

from oracle import fhgs_oracle as fo
from paper_2505_19154_b200 import inputs

C0 = 0.28209479177387814
SURFEL = fo.params(primitive=1)


def cam35(cam):
    return fo.cam_array(cam.view, cam.proj, cam.cam_pos)


def project_surfels(mean, scale, quat, opacity, cam, colour=(0.2, 0.4, 0.6), params=SURFEL):
    mean = np.atleast_2d(np.asarray(mean, np.float32))
    n = mean.shape[0]
    scale = np.broadcast_to(np.asarray(scale, np.float32), (n, 3)).copy()
    quat = np.broadcast_to(np.asarray(quat, np.float32), (n, 4)).copy()
    opacity = np.broadcast_to(np.asarray(opacity, np.float32), (n,)).copy()
    sh = ((np.broadcast_to(np.asarray(colour, np.float64), (n, 3)) - 0.5) / C0).astype(np.float32).reshape(n, 1, 3)
    return fo.project(mean, scale, quat, opacity, sh, 0, cam35(cam), cam.width, cam.height, params)


def uv(pr, i, x, y):
    p, num, den = fo.surfel_terms(pr["ray_transform"][i], x, y)
    return float(p[0]) / float(p[2]), float(p[1]) / float(p[2]), num / den


def quat_rot(q):
    """Rotation matrix of a unit quaternion (w,x,y,z), Hamilton convention, float64 -- written out here."""
    w, x, y, z = np.asarray(q, np.float64) / np.linalg.norm(q)
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                     [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                     [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])


def pinhole(cam, P):
    """Independent pinhole: world point -> continuous pixel coordinates and camera depth (float64)."""
    V = cam.view.astype(np.float64).reshape(4, 4)
    pr = cam.proj.astype(np.float64).reshape(4, 4)
    c = V[:3, :3] @ P + V[:3, 3]
    fx, fy = pr[0, 0] * cam.width / 2, pr[1, 1] * cam.height / 2
    cx, cy = (pr[0, 2] + 1) * cam.width / 2 - 0.5, (pr[1, 2] + 1) * cam.height / 2 - 0.5
    return fx * c[0] / c[2] + cx, fy * c[1] / c[2] + cy, c[2]


def test_spec_worked_intersections():
    """camera at the origin looking +z, frontal unit splat in the plane z = 1: the central ray hits
    (u,v) = (0,0), G = 1; with the splat shifted to p = (0.5, 0, 1) it hits (u,v) = (-0.5, 0), G = e^-0.125 = 0.8825."""
    cam = inputs.look_at_camera((0, 0, 0), (0, 0, 1), 65, 65)        # principal point = pixel (32, 32)
    pr = project_surfels([(0, 0, 1), (0.5, 0, 1)], (1, 1, 1), (1, 0, 0, 0), 0.7, cam)
    u, v, q = uv(pr, 0, 32, 32)
    assert abs(u) < 1e-6 and abs(v) < 1e-6 and q < 1e-10
    u, v, q = uv(pr, 1, 32, 32)
    assert abs(u + 0.5) < 1e-6 and abs(v) < 1e-6 and abs(math.exp(-0.5 * q) - 0.8825) < 5e-5
    assert abs(float(pr["depth"][0]) - 1.0) < 1e-7
    # one pixel to the right: the ray direction is ((x - cx)/fx, 0, 1), so u = 1/fx on the z = 1 plane
    fx = (65 / 2) / math.tan(math.radians(30))
    u, v, q = uv(pr, 0, 33, 32)
    assert abs(u - 1 / fx) < 1e-6 and abs(v) < 1e-6
    # rendering that single splat: alpha = op * G at the centre, T = 1 - alpha
    order = fo.global_order(pr)[:1]
    out = fo.render_literal({k: (v[:1] if k != "ray_transform" else v[:1]) for k, v in pr.items()}, order, None, 65, 65,
                            SURFEL, pix=np.array([32 * 65 + 32], np.int32))
    assert abs(out["T"][0] - 0.3) < 1e-6 and out["n"][0] == 1


def test_scales_and_tangent_frame():
    """Eq. 2: P(u,v) = p + s_u t_u u + s_v t_v v with t_u, t_v the first two columns of R(quat).  For random splats and
    pixels the (u,v) returned by the oracle, pushed through Eq. 2 and an independent float64 pinhole, lands on the query
    pixel (SPEC.md:142 asks 1e-4 px in double; the ray transform is binary32, hence 5e-3 px)."""
    rng = np.random.default_rng(3)
    cam = inputs.look_at_camera((0.3, -0.2, -4.0), (0.1, 0.0, 0.2), 96, 80)
    n = 300
    mean = rng.uniform(-1, 1, (n, 3)).astype(np.float32)
    scale = np.exp(rng.normal(-1.5, 0.5, (n, 3))).astype(np.float32)
    quat = rng.normal(size=(n, 4)).astype(np.float32)
    pr = fo.project(mean, scale, quat, np.full(n, 0.5, np.float32), np.zeros((n, 1, 3), np.float32), 0, cam35(cam), 96, 80, SURFEL)
    checked = 0
    for i in np.nonzero(pr["radius"] > 0)[0][:150]:
        R = quat_rot(quat[i])
        for _ in range(4):
            x = int(np.clip(round(float(pr["xy"][i, 0]) + rng.integers(-3, 4)), 0, 95))
            y = int(np.clip(round(float(pr["xy"][i, 1]) + rng.integers(-3, 4)), 0, 79))
            u, v, q = uv(pr, i, x, y)
            if not q <= 9.0:
                continue
            P = mean[i].astype(np.float64) + scale[i, 0] * R[:, 0] * u + scale[i, 1] * R[:, 1] * v
            X, Y, z = pinhole(cam, P)
            assert abs(X - x) < 5e-3 and abs(Y - y) < 5e-3 and z > 0.2, (i, x, y, X, Y)
            checked += 1
    assert checked > 200


def test_screen_bounds_conservative_and_sized():
    """frontal unit splat at depth 1 with fx = fy = 100 spans >= 600 px; and, by exhaustive scan over
    64x64 images, no pixel with u^2+v^2 <= 9 lies outside the rectangle / the radius box of its splat."""
    W = 200
    fov = 2 * math.degrees(math.atan((W / 2) / 100.0))
    cam = inputs.look_at_camera((0, 0, 0), (0, 0, 1), W, W, fov_x_deg=fov)
    pr = project_surfels((0, 0, 4.0), (1, 1, 1), (1, 0, 0, 0), 0.5, cam)      # depth 4: half extent 3 * 100 / 4 = 75 px
    assert 75 <= float(pr["conic_opacity"][0, 0]) <= 77.5 and 75 <= float(pr["conic_opacity"][0, 1]) <= 77.5
    near = fo.params(primitive=1, z_near=0.01)
    pr1 = project_surfels((0, 0, 1.0), (0.3, 0.3, 1), (1, 0, 0, 0), 0.5, cam, params=near)   # 3 sigma = 0.9 at depth 1 -> 90 px
    assert 90 <= float(pr1["conic_opacity"][0, 0]) <= 92.5
    rng = np.random.default_rng(11)
    cam = inputs.look_at_camera((0, 0, -4.0), (0, 0, 0), 64, 64)
    n = 400
    mean = rng.uniform(-1.2, 1.2, (n, 3)).astype(np.float32)
    scale = np.exp(rng.normal(-2.0, 0.8, (n, 3))).astype(np.float32)
    quat = rng.normal(size=(n, 4)).astype(np.float32)
    pr = fo.project(mean, scale, quat, np.full(n, 0.5, np.float32), np.zeros((n, 1, 3), np.float32), 0, cam35(cam), 64, 64, SURFEL)
    seen = 0
    for i in np.nonzero(pr["radius"] > 0)[0]:
        rt = pr["ray_transform"][i].astype(np.float64)
        ys, xs = np.mgrid[0:64, 0:64]
        px = xs * rt[0] + ys * rt[1] + rt[2]
        py = xs * rt[4] + ys * rt[5] + rt[6]
        pz = xs * rt[8] + ys * rt[9] + rt[10]
        inside = (px * px + py * py) <= (9.0 + 1e-3) * pz * pz
        inside &= pz != 0
        if not inside.any():
            continue
        seen += 1
        r = float(pr["radius"][i])
        assert np.all(np.abs(xs[inside] - pr["xy"][i, 0]) <= r) and np.all(np.abs(ys[inside] - pr["xy"][i, 1]) <= r)
        x0, y0, x1, y1 = pr["rect"][i].astype(int)
        tx, ty = xs[inside] // 16, ys[inside] // 16
        assert np.all((tx >= x0) & (tx < x1) & (ty >= y0) & (ty < y1))
    assert seen > 200


def test_culling_cases():
    cam = inputs.look_at_camera((0, 0, 0), (0, 0, 1), 64, 64)
    # behind the camera; in front but its 3-sigma disc crosses the near plane; well in front
    tilt = (math.cos(math.radians(40)), 0.0, math.sin(math.radians(40)), 0.0)     # rotation about y: the disc dips towards the camera
    pr = project_surfels([(0, 0, -1.0), (0, 0, 1.0), (0, 0, 4.0)], (0.6, 0.6, 1), [(1, 0, 0, 0), tilt, tilt], 0.5, cam)
    assert pr["radius"].tolist()[0] == 0 and pr["tiles_touched"][0] == 0
    assert pr["radius"][1] == 0, "z_min = 1 - 3*0.6*sin(80deg) < z_near"
    assert pr["radius"][2] > 0
    assert np.all(pr["ray_transform"][:2] == 0)
    # a splat seen exactly edge-on has an empty footprint: nothing may be blended anywhere
    edge = (math.cos(math.radians(45)), 0.0, math.sin(math.radians(45)), 0.0)      # t_u along -z, t_v along y: normal = x axis
    pr = project_surfels((0, 0, 4.0), (0.1, 0.1, 1), edge, 0.9, cam)
    order = fo.global_order(pr)
    out = fo.render_literal(pr, order, None, 64, 64, SURFEL)
    assert out["n"].sum() <= 64            # at most one pixel column (the line the disc projects to)


def test_small_splat_limit_matches_ewa():
    """Independent cross-check of the whole chain: for a small splat the perspective map is affine over its footprint,
    and the surfel density equals the EWA density of the flat Gaussian (third scale -> 0) without the 0.3 px^2 dilation."""
    rng = np.random.default_rng(5)
    cam = inputs.look_at_camera((0.0, 0.0, -20.0), (0, 0, 0), 128, 128, fov_x_deg=10.0)   # far and narrow: nearly affine
    n = 60
    mean = rng.uniform(-0.4, 0.4, (n, 3)).astype(np.float32)
    scale = np.concatenate([np.exp(rng.normal(-3.2, 0.3, (n, 2))), np.full((n, 1), 1e-6)], axis=1).astype(np.float32)
    quat = (np.array([1, 0, 0, 0]) + 0.25 * rng.normal(size=(n, 4))).astype(np.float32)   # moderately tilted
    op = np.full(n, 0.5, np.float32)
    sh = np.zeros((n, 1, 3), np.float32)
    ps = fo.project(mean, scale, quat, op, sh, 0, cam35(cam), 128, 128, SURFEL)
    pe = fo.project(mean, scale, quat, op, sh, 0, cam35(cam), 128, 128, fo.params(cov_dilation=0.0))
    worst = 0.0
    cnt = 0
    for i in range(n):
        if ps["radius"][i] == 0 or pe["radius"][i] == 0:
            continue
        cx, cy = pe["xy"][i]
        for dx in (-2, 0, 1, 3):
            for dy in (-1, 0, 2):
                x, y = int(round(cx)) + dx, int(round(cy)) + dy
                qe = fo.q_value(cx, cy, *pe["conic_opacity"][i, :3], x, y)
                _, _, qs = uv(ps, i, x, y)
                if qe <= 9.0:
                    worst = max(worst, abs(math.exp(-0.5 * qe) - math.exp(-0.5 * qs)))
                    cnt += 1
    assert cnt > 200 and worst < 5e-3, worst


def test_rigid_motion_invariance():
    """Moving camera and splats together leaves (u, v) unchanged (SPEC.md: intersect is invariant under rigid motion)."""
    rng = np.random.default_rng(8)
    n = 50
    mean = rng.uniform(-0.8, 0.8, (n, 3))
    scale = np.exp(rng.normal(-2.0, 0.4, (n, 3))).astype(np.float32)
    quat = rng.normal(size=(n, 4))
    quat /= np.linalg.norm(quat, axis=1, keepdims=True)
    cam0 = inputs.look_at_camera((0, 0, -4.0), (0, 0, 0), 64, 64)
    # rigid motion: rotation Q (from a quaternion qm) and translation t
    qm = np.array([0.9, 0.2, -0.3, 0.1]); qm /= np.linalg.norm(qm)
    Q = quat_rot(qm)
    t = np.array([0.7, -1.1, 0.4])

    def qmul(a, b):
        w1, x1, y1, z1 = a; w2, x2, y2, z2 = b
        return np.array([w1 * w2 - x1 * x2 - y1 * y2 - z1 * z2, w1 * x2 + x1 * w2 + y1 * z2 - z1 * y2,
                         w1 * y2 - x1 * z2 + y1 * w2 + z1 * x2, w1 * z2 + x1 * y2 - y1 * x2 + z1 * w2])
    mean1 = mean @ Q.T + t
    quat1 = np.array([qmul(qm, q) for q in quat])
    V0 = cam0.view.astype(np.float64).reshape(4, 4)
    M = np.eye(4); M[:3, :3] = Q; M[:3, 3] = t
    V1 = V0 @ np.linalg.inv(M)
    pos1 = Q @ cam0.cam_pos.astype(np.float64) + t
    cam1 = inputs.Camera(V1.astype(np.float32).reshape(16), cam0.proj, pos1.astype(np.float32), 64, 64)
    sh = np.zeros((n, 1, 3), np.float32); op = np.full(n, 0.5, np.float32)
    p0 = fo.project(mean.astype(np.float32), scale, quat.astype(np.float32), op, sh, 0, cam35(cam0), 64, 64, SURFEL)
    p1 = fo.project(mean1.astype(np.float32), scale, quat1.astype(np.float32), op, sh, 0, cam35(cam1), 64, 64, SURFEL)
    cnt = 0
    for i in range(n):
        if p0["radius"][i] == 0 or p1["radius"][i] == 0:
            continue
        x, y = int(round(float(p0["xy"][i, 0]))), int(round(float(p0["xy"][i, 1])))
        u0, v0, q0 = uv(p0, i, x, y)
        u1, v1, q1 = uv(p1, i, x, y)
        if q0 <= 9:
            assert abs(u0 - u1) < 2e-4 and abs(v0 - v1) < 2e-4
            cnt += 1
    assert cnt > 20


def _tiny_surfel(view=0, n=600):
    cfg = inputs.scaled(inputs.CONFIGS["tiny"], n=n, log_scale_mu=-2.2)
    sc = inputs.make_scene(cfg)
    cam = inputs.make_camera(cfg, view)
    pr = fo.project(sc.mean, sc.scale, sc.quat, sc.opacity, sc.sh, sc.sh_degree, cam35(cam), 64, 64, SURFEL)
    return cfg, sc, cam, pr


def test_literal_equals_scatter_and_invariants():
    """Surfel mode through the unchanged drivers: literal == scatter bitwise; sum of weights = 1 - T; a constant feature
    renders to (1 - T) * constant; a constant GT map fuses to the constant; bins are consistent with the rectangles."""
    cfg, sc, cam, pr = _tiny_surfel(1)
    assert (pr["radius"] > 0).sum() > 300
    order = fo.global_order(pr)
    feat = np.ones((sc.n, 4), np.float32) * np.array([1.0, -2.0, 0.5, 3.0], np.float32)
    a = fo.render_literal(pr, order, feat, 64, 64, SURFEL)
    b = fo.render_scatter(pr, order, feat, 64, 64, SURFEL)
    for key in ("rgb", "feat", "T", "n", "fragile"):
        assert np.array_equal(a[key], b[key]), key
    assert a["n"].max() > 5
    np.testing.assert_allclose(a["feat"], (1.0 - a["T"])[:, None] * np.array([1.0, -2.0, 0.5, 3.0]), atol=1e-12)
    gt = np.broadcast_to(np.array([0.25, -1.0, 2.0, 0.5], np.float32), (64, 64, 4)).copy()
    n1, d1 = fo.fuse(pr, order, gt, 64, 64, SURFEL, literal=True)
    n2, d2 = fo.fuse(pr, order, gt, 64, 64, SURFEL, literal=False)
    np.testing.assert_allclose(n2, n1, rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(d1.sum(), (1.0 - a["T"]).sum(), rtol=1e-10)           # conservation
    seen = d1 > 1e-8
    np.testing.assert_allclose(n1[seen] / d1[seen, None], np.broadcast_to(gt[0, 0], (int(seen.sum()), 4)), atol=1e-9)
    bo = fo.bins(pr, 64, 64)
    assert bo["M"] == int(pr["tiles_touched"].sum())
    # the EWA state of the same scene is a different image: the mode switch is not a no-op
    pe = fo.project(sc.mean, sc.scale, sc.quat, sc.opacity, sc.sh, sc.sh_degree, cam35(cam), 64, 64)
    e = fo.render_literal(pe, fo.global_order(pe), None, 64, 64)
    assert np.abs(e["T"] - a["T"]).max() > 0.05


def test_ndfd_on_surfels_forward_identities_and_backward_finite_differences():
    """The NDFD oracle over surfels: O(N) recurrence == explicit pair sum in both accumulation orders, k = 0 closed form
    against the surfel renderer, and dL/d opacity == central finite differences of the forward oracle."""
    cfg, sc, cam, pr = _tiny_surfel(3)
    order = fo.global_order(pr)
    rng = np.random.default_rng(31)
    feat = rng.standard_normal((sc.n, 12)).astype(np.float32)
    feat /= np.linalg.norm(feat, axis=1, keepdims=True)
    gt = rng.standard_normal((64, 64, 12)).astype(np.float32)
    gt /= np.linalg.norm(gt, axis=2, keepdims=True)
    pix = np.arange(0, 64 * 64, 7, dtype=np.int32)
    for mode in (0, 1):
        lgt, lcf, pw = fo.ndfd(pr, order, feat, gt, 64, 64, mode=mode, params=SURFEL, pix=pix, pairwise=True)
        np.testing.assert_allclose(lcf, pw, rtol=1e-9, atol=1e-12)
    r = fo.render_literal(pr, order, feat, 64, 64, SURFEL, pix=pix)
    lgt0, lcf0 = fo.ndfd(pr, order, feat, gt, 64, 64, k=0.0, params=SURFEL, pix=pix)
    Ws = 1.0 - r["T"]
    np.testing.assert_allclose(lgt0, 0.5 * Ws, atol=1e-12)
    np.testing.assert_allclose(lcf0, 0.25 * (Ws ** 2 - (r["feat"] ** 2).sum(axis=1)), atol=2e-7)   # features are unit-norm to fp32 rounding
    prm = SURFEL.copy()
    prm[5] = 0.0            # t_min = 0: the fragment lists do not change under the perturbation
    lam1, lam2 = 0.7, 1.3
    L, grad = fo.ndfd_backward(pr, order, feat, gt, 64, 64, lam1=lam1, lam2=lam2, params=prm)

    def forward_total(p):
        a, b = fo.ndfd(p, order, feat, gt, 64, 64, params=prm)
        return lam1 * a.sum() + lam2 * b.sum()

    assert abs(L - forward_total(pr)) <= 1e-9 * abs(L)
    probe = np.argsort(-np.abs(grad))[[0, 1, 3, 10, 40]]
    assert np.abs(grad[probe]).min() > 0
    for g in probe:
        o0 = pr["conic_opacity"][g, 3]
        hi, lo = np.float32(o0 * (1 + 2e-3)), np.float32(o0 * (1 - 2e-3))
        p_hi = dict(pr, conic_opacity=pr["conic_opacity"].copy()); p_hi["conic_opacity"][g, 3] = hi
        p_lo = dict(pr, conic_opacity=pr["conic_opacity"].copy()); p_lo["conic_opacity"][g, 3] = lo
        fd = (forward_total(p_hi) - forward_total(p_lo)) / (float(hi) - float(lo))
        assert abs(fd - grad[g]) <= 2e-4 * max(abs(grad[g]), 1e-3), (g, fd, grad[g])

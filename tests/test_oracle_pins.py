"""Pins for the CPU oracle: closed forms, worked values, invariants and brute
force that a plausible mistake in oracle/fhgs_oracle.c would fail.  CPU only."""
import math

import numpy as np
import pytest

from oracle import fhgs_oracle as fo
from paper_2505_19154_b200 import inputs

C0 = 0.28209479177387814


def cam35(cam):
    return fo.cam_array(cam.view, cam.proj, cam.cam_pos)


def front_camera(w, h):
    return inputs.look_at_camera((0.0, 0.0, 0.0), (0.0, 0.0, 1.0), w, h)


def scene_arrays(mean, scale, quat, opacity, colour):
    mean = np.atleast_2d(np.asarray(mean, np.float32))
    n = mean.shape[0]
    scale = np.broadcast_to(np.asarray(scale, np.float32), (n, 3)).copy()
    quat = np.broadcast_to(np.asarray(quat, np.float32), (n, 4)).copy()
    opacity = np.broadcast_to(np.asarray(opacity, np.float32), (n,)).copy()
    colour = np.broadcast_to(np.asarray(colour, np.float64), (n, 3))
    sh = ((colour - 0.5) / C0).astype(np.float32).reshape(n, 1, 3)
    return mean, scale, quat, opacity, sh


def project_simple(mean, scale, quat, opacity, colour, cam, params=fo.DEFAULT_PARAMS):
    m, s, q, o, sh = scene_arrays(mean, scale, quat, opacity, colour)
    return fo.project(m, s, q, o, sh, 0, cam35(cam), cam.width, cam.height, params)


def manual_pr(xy, conic, opac, rgb, radius):
    """Hand-made projected state to pin compositing independently of projection."""
    xy = np.atleast_2d(np.asarray(xy, np.float32))
    n = xy.shape[0]
    co = np.zeros((n, 4), np.float32)
    co[:, :3] = np.asarray(conic, np.float32)
    co[:, 3] = np.asarray(opac, np.float32)
    return dict(xy=xy, conic_opacity=co,
                rgb=np.broadcast_to(np.asarray(rgb, np.float32), (n, 3)).copy(),
                radius=np.broadcast_to(np.asarray(radius, np.int32), (n,)).copy(),
                depth=np.arange(1, n + 1, dtype=np.float32))


def tiny_state(view=0, n=None):
    cfg = inputs.CONFIGS["tiny"]
    if n is not None:
        cfg = inputs.scaled(cfg, n=n)
    sc = inputs.make_scene(cfg)
    cam = inputs.make_camera(cfg, view)
    pr = fo.project(sc.mean, sc.scale, sc.quat, sc.opacity, sc.sh, sc.sh_degree, cam35(cam),
                    cam.width, cam.height)
    return cfg, sc, cam, pr


# ---- C3-1: isotropic Gaussian on the optical axis ------------------------------------------------
def test_pin01_isotropic_on_axis_footprint():
    cam = front_camera(64, 64)
    rng = np.random.default_rng(0)
    quat = rng.standard_normal(4)
    pr = project_simple([0, 0, 4.0], [0.1, 0.1, 0.1], quat, 0.7, [0.2, 0.4, 0.6], cam)
    fx = 32.0 / math.tan(math.radians(30.0))
    assert abs(fx - 55.425626) < 1e-5                      # SURVEY appendix A worked value
    a = (fx * 0.1 / 4.0) ** 2 + 0.3
    assert abs(a - 2.2200) < 1e-4
    np.testing.assert_allclose(pr["xy"][0], [31.5, 31.5], atol=1e-5)
    np.testing.assert_allclose(pr["conic_opacity"][0], [1 / a, 0.0, 1 / a, 0.7], rtol=2e-6, atol=2e-7)
    assert abs(pr["conic_opacity"][0, 0] - 0.450450) < 1e-5
    assert pr["radius"][0] == 5 == math.ceil(3 * math.sqrt(a))
    assert abs(pr["depth"][0] - 4.0) < 1e-6
    # rect: px +- r = [26.5, 36.5] -> tiles 1..2 in x and y
    assert pr["rect"][0].tolist() == [1, 1, 3, 3] and pr["tiles_touched"][0] == 4
    np.testing.assert_allclose(pr["rgb"][0], [0.2, 0.4, 0.6], atol=1e-6)
    # pixel (31,31) is at d = (1/2, 1/2): q = 0.5/a, G = exp(-q/2)
    q = fo.q_value(*pr["xy"][0], *pr["conic_opacity"][0, :3], 31, 31)
    assert abs(q - 0.225225) < 1e-5
    order = fo.global_order(pr)
    out = fo.render_literal(pr, order, None, 64, 64, pix=np.array([31 * 64 + 31]))
    G = math.exp(-q / 2)
    assert abs(G - 0.893497) < 1e-5
    assert abs(out["T"][0] - (1 - 0.7 * G)) < 1e-6
    np.testing.assert_allclose(out["rgb"][0], 0.7 * G * np.array([0.2, 0.4, 0.6]), atol=1e-6)


# ---- C3-2: off-axis closed form ------------------------------------------------------------------
def test_pin02_off_axis_covariance():
    cam = front_camera(64, 64)
    fx = 32.0 / math.tan(math.radians(30.0))
    X, z, s = 1.0, 4.0, 0.1          # u = 0.25 < 1.3*tan(30deg): clamp inactive
    pr = project_simple([X, 0, z], [s, s, s], [1, 0, 0, 0], 0.5, [0.5, 0.5, 0.5], cam)
    a = (fx * s / z) ** 2 * (1 + (X / z) ** 2) + 0.3
    c = (fx * s / z) ** 2 + 0.3
    det = a * c
    np.testing.assert_allclose(pr["conic_opacity"][0, :3], [c / det, 0.0, a / det], rtol=1e-5, atol=1e-6)
    np.testing.assert_allclose(pr["xy"][0], [fx * X / z + 31.5, 31.5], rtol=1e-6)


def _quat_rotate(q, v):
    """v' = q v q* by Hamilton products (independent of the matrix formula)."""
    q = np.asarray(q, np.float64)
    q = q / np.linalg.norm(q)

    def mul(a, b):
        return np.array([a[0]*b[0] - a[1]*b[1] - a[2]*b[2] - a[3]*b[3],
                         a[0]*b[1] + a[1]*b[0] + a[2]*b[3] - a[3]*b[2],
                         a[0]*b[2] - a[1]*b[3] + a[2]*b[0] + a[3]*b[1],
                         a[0]*b[3] + a[1]*b[2] - a[2]*b[1] + a[3]*b[0]])
    qc = q * np.array([1, -1, -1, -1.0])
    return mul(mul(q, np.array([0.0, *v])), qc)[1:]


def test_pin02b_general_covariance_by_finite_differences():
    """Anisotropic, rotated Gaussians seen by a rotated camera: Sigma2D = sum_k (d pi . a_k)(...)^T
    with the 3 semi-axes a_k = s_k * (q e_k q*) pushed through the pinhole map by central
    differences in float64 -- no matrix from the oracle's own derivation is reused."""
    cfg = inputs.CONFIGS["tiny"]
    cam = inputs.make_camera(cfg, 1)
    rng = np.random.default_rng(5)
    n = 40
    mean = rng.uniform(-1, 1, (n, 3)).astype(np.float32)
    scale = np.exp(rng.normal(-3, 0.5, (n, 3))).astype(np.float32)
    quat = rng.standard_normal((n, 4)).astype(np.float32)
    m, s, q, o, sh = scene_arrays(mean, scale, quat, 0.5, [0.5, 0.5, 0.5])
    s[:] = scale
    q[:] = quat
    pr = fo.project(m, s, q, o, sh, 0, cam35(cam), 64, 64)
    V = cam.view.astype(np.float64).reshape(4, 4)
    fx = 32.0 / math.tan(math.radians(30.0))

    def pinhole(pw):
        t = V[:3, :3] @ pw + V[:3, 3]
        return np.array([fx * t[0] / t[2] + 31.5, fx * t[1] / t[2] + 31.5]), t[2]
    checked = 0
    for i in range(n):
        if pr["radius"][i] == 0:
            continue
        p = mean[i].astype(np.float64)
        centre, z = pinhole(p)
        t = V[:3, :3] @ p + V[:3, 3]
        if abs(t[0] / t[2]) > 1.3 * math.tan(math.radians(30)) or abs(t[1] / t[2]) > 1.3 * math.tan(math.radians(30)):
            continue                                          # Jacobian clamp active: not this pin
        cov = np.zeros((2, 2))
        for k in range(3):
            a = scale[i, k].astype(np.float64) * _quat_rotate(quat[i], np.eye(3)[k])
            eps = 1e-6
            d = (pinhole(p + eps * a / np.linalg.norm(a))[0] - pinhole(p - eps * a / np.linalg.norm(a))[0]) / (2 * eps)
            d = d * np.linalg.norm(a)
            cov += np.outer(d, d)
        cov += 0.3 * np.eye(2)
        con = np.linalg.inv(cov)
        np.testing.assert_allclose(pr["xy"][i], centre, rtol=1e-5, atol=1e-4)
        np.testing.assert_allclose(pr["conic_opacity"][i, :3], [con[0, 0], con[0, 1], con[1, 1]],
                                   rtol=2e-4, atol=2e-5)
        lam = np.linalg.eigvalsh(cov).max()
        assert abs(pr["radius"][i] - math.ceil(3 * math.sqrt(lam))) <= (1 if abs(3 * math.sqrt(lam) % 1) < 1e-4 else 0)
        assert abs(pr["depth"][i] - z) < 1e-5
        checked += 1
    assert checked >= 20


# ---- C3-3: two-Gaussian compositing --------------------------------------------------------------
def test_pin03_two_gaussian_compositing():
    cam = front_camera(65, 65)        # cx = cy = 32: pixel (32,32) is exactly at the splat centre
    pr = project_simple([[0, 0, 2.0], [0, 0, 3.0]], [0.2, 0.2, 0.2], [1, 0, 0, 0], 0.5,
                        [[1, 0, 0], [0, 0, 1]], cam)
    order = fo.global_order(pr)
    assert order.tolist() == [0, 1]
    feat = np.array([[1.0, 0.0], [0.0, 1.0]], np.float32)   # channel k carries w_k
    out = fo.render_literal(pr, order, feat, 65, 65, pix=np.array([32 * 65 + 32]))
    np.testing.assert_allclose(out["feat"][0], [0.5, 0.25], atol=1e-7)         # w = (0.5, 0.25)
    np.testing.assert_allclose(out["rgb"][0], [0.5, 0.0, 0.25], atol=1e-6)
    assert abs(out["T"][0] - 0.25) < 1e-7 and out["n"][0] == 2
    # with background bg: C + T*bg
    prm = fo.DEFAULT_PARAMS.copy()
    prm[7:10] = [0.2, 0.4, 0.8]
    out = fo.render_literal(pr, order, None, 65, 65, params=prm, pix=np.array([32 * 65 + 32]))
    np.testing.assert_allclose(out["rgb"][0], np.array([0.5, 0.0, 0.25]) + 0.25 * prm[7:10], atol=1e-6)
    # far-first order would give (0.25, 0, 0.5): the nearest occludes (reading C2-1)
    assert out["rgb"][0][0] > out["rgb"][0][2]


# ---- C3-4: G values and the cut-off edge ----------------------------------------------------------
def test_pin04_gaussian_values_and_cutoff():
    for d, G in [(0.0, 1.0), (1.0, 0.606531), (3.0, 0.011109)]:
        pr = manual_pr([d, 0.0], [1.0, 0.0, 1.0], 1.0 if d else 0.5, [1, 1, 1], 5)
        out = fo.render_literal(pr, np.array([0], np.uint32), None, 4, 4, pix=np.array([0]))
        alpha = (1.0 if d else 0.5) * G
        assert out["n"][0] == 1
        assert abs((1 - out["T"][0]) - alpha) < 1e-6
    # q == 9 exactly is included, the next float above is not ("G < e^-4.5 ignored")
    assert fo.q_value(3.0, 0.0, 1.0, 0.0, 1.0, 0, 0) == 9.0
    pr = manual_pr([np.nextafter(np.float32(3.0), np.float32(4.0)), 0.0], [1.0, 0.0, 1.0], 1.0, [1, 1, 1], 5)
    out = fo.render_literal(pr, np.array([0], np.uint32), None, 4, 4, pix=np.array([0]))
    assert out["n"][0] == 0 and out["T"][0] == 1.0
    # cross term: q = A dx^2 + 2 B dx dy + C dy^2 with d = centre - pixel
    q = fo.q_value(2.0, 3.0, 0.5, 0.25, 0.75, 1, 1)    # dx = 1, dy = 2
    assert abs(q - (0.5 * 1 + 2 * 0.25 * 2 + 0.75 * 4)) < 1e-6
    q = fo.q_value(0.0, 3.0, 0.5, 0.25, 0.75, 1, 1)    # dx = -1, dy = 2: cross term flips sign
    assert abs(q - (0.5 * 1 - 2 * 0.25 * 2 + 0.75 * 4)) < 1e-6


# ---- C3-5: opaque fragment, clamp and stop interplay ----------------------------------------------
def test_pin05_opaque_fragment_clamp():
    pr = manual_pr([[0, 0], [0, 0], [0, 0]], [1.0, 0.0, 1.0], [1.0, 1.0, 1.0],
                   [[1, 0, 0], [0, 1, 0], [0, 0, 1]], 5)
    out = fo.render_literal(pr, np.array([0, 1, 2], np.uint32), None, 4, 4, pix=np.array([0]))
    amax = float(np.float32(0.9999))
    # after the first: T = 1 - 0.9999f = 1.00017e-4 >= t_min -> the second IS blended; then T < t_min
    assert abs((1 - amax) - 1.00016594e-4) < 1e-11
    assert out["n"][0] == 2
    np.testing.assert_allclose(out["rgb"][0], [amax, (1 - amax) * amax, 0.0], atol=1e-12)
    assert abs(out["T"][0] - (1 - amax) ** 2) < 1e-15
    assert out["fragile"][0] == 0          # |T/t_min - 1| = 1.7e-4 is outside the fragile band


# ---- C3-6/7: sum of weights, transmittance, constant features -------------------------------------
def test_pin06_07_weight_sum_and_constant_feature():
    cfg, sc, cam, pr = tiny_state(0)
    order = fo.global_order(pr)
    v = np.array([0.3, -1.2, 2.0], np.float32)
    feat = np.broadcast_to(v, (sc.n, 3)).copy()
    out = fo.render_literal(pr, order, feat, 64, 64)
    assert np.all(out["T"] <= 1.0) and np.all(out["T"] >= 0.0)
    np.testing.assert_allclose(out["feat"], (1 - out["T"])[:, None] * v[None, :].astype(np.float64), atol=1e-12)
    assert (out["n"] > 0).sum() > 500


def test_pin06b_empty_scene_is_background():
    prm = fo.DEFAULT_PARAMS.copy()
    prm[7:10] = [0.1, 0.2, 0.3]
    pr = manual_pr(np.zeros((0, 2)), np.zeros((0, 3)), np.zeros(0), np.zeros((0, 3)), np.zeros(0))
    out = fo.render_literal(pr, np.zeros(0, np.uint32), None, 8, 8, params=prm)
    np.testing.assert_allclose(out["rgb"], np.broadcast_to(prm[7:10].astype(np.float64), (64, 3)))
    assert np.all(out["T"] == 1.0) and np.all(out["n"] == 0)
    out = fo.render_scatter(pr, np.zeros(0, np.uint32), None, 8, 8, params=prm)
    np.testing.assert_allclose(out["rgb"], np.broadcast_to(prm[7:10].astype(np.float64), (64, 3)))


# ---- C3-8: a constant GT map fuses to that constant -----------------------------------------------
def test_pin08_constant_map_fuses_to_constant():
    cfg, sc, cam, pr = tiny_state(1)
    order = fo.global_order(pr)
    v = np.array([0.5, -2.0, 3.25, 0.0], np.float32)
    gt = np.broadcast_to(v, (64, 64, 4)).copy()
    for literal in (True, False):
        num, den = fo.fuse(pr, order, gt, 64, 64, literal=literal)
        prev = np.full((sc.n, 4), 7.0)
        f = fo.finalize(num, den, prev)
        covered = den > 1e-8
        assert covered.sum() > 300
        np.testing.assert_allclose(f[covered], np.broadcast_to(v.astype(np.float64), (covered.sum(), 4)), rtol=1e-12)
        assert np.all(f[~covered] == 7.0)            # unseen Gaussians keep their feature (C2-17)
        fn = fo.finalize(num, den, prev, l2norm=True)
        np.testing.assert_allclose(np.linalg.norm(fn[covered], axis=1), 1.0, rtol=1e-12)


# ---- C3-9: conservation, C3-10: adjointness -------------------------------------------------------
def test_pin09_10_conservation_and_adjointness():
    cfg, sc, cam, pr = tiny_state(2)
    order = fo.global_order(pr)
    rng = np.random.default_rng(3)
    D = 5
    gt = rng.standard_normal((64, 64, D)).astype(np.float32)
    feat = rng.standard_normal((sc.n, D)).astype(np.float32)
    out = fo.render_literal(pr, order, feat, 64, 64)
    num, den = fo.fuse(pr, order, gt, 64, 64, literal=True)
    cover = 1.0 - out["T"]
    assert abs(den.sum() - cover.sum()) < 1e-9 * cover.sum()
    np.testing.assert_allclose(num.sum(axis=0), (cover[:, None] * gt.reshape(-1, D)).sum(axis=0), rtol=1e-9, atol=1e-9)
    lhs = (out["feat"] * gt.reshape(-1, D)).sum()
    rhs = (feat.astype(np.float64) * num).sum()
    assert abs(lhs - rhs) < 1e-9 * max(1.0, abs(lhs))


# ---- C3-11: single Gaussian, no occlusion: brute-force weighted mean ------------------------------
def test_pin11_single_gaussian_fusion_bruteforce():
    cam = front_camera(64, 64)
    pr = project_simple([0.3, -0.2, 3.0], [0.25, 0.1, 0.05], [0.9, 0.1, 0.3, -0.2], 0.8, [0.5, 0.5, 0.5], cam)
    assert pr["radius"][0] > 0
    rng = np.random.default_rng(11)
    gt = rng.standard_normal((64, 64, 3)).astype(np.float32)
    num, den = fo.fuse(pr, fo.global_order(pr), gt, 64, 64, literal=True)
    A, B, Cc, o = pr["conic_opacity"][0].astype(np.float64)
    ys, xs = np.mgrid[0:64, 0:64]
    dx = pr["xy"][0, 0].astype(np.float64) - xs
    dy = pr["xy"][0, 1].astype(np.float64) - ys
    q = A * dx * dx + 2 * B * dx * dy + Cc * dy * dy
    w = np.where(q <= 9.0, np.minimum(0.9999, o * np.exp(-q / 2)), 0.0)
    # pixels within 1e-4 of the cut-off may fall either side in fp32: exclude by construction
    assert np.all(np.abs(q - 9.0) > 1e-4)
    np.testing.assert_allclose(den[0], w.sum(), rtol=1e-5)
    np.testing.assert_allclose(num[0], (w[..., None] * gt).sum(axis=(0, 1)), rtol=1e-4, atol=1e-5)
    f = fo.finalize(num, den, np.zeros((1, 3)))
    np.testing.assert_allclose(f[0], (w[..., None] * gt).sum(axis=(0, 1)) / w.sum(), rtol=1e-4, atol=1e-5)
    num2, den2 = fo.fuse(pr, fo.global_order(pr), gt, 64, 64, literal=False)
    np.testing.assert_allclose(num2, num, rtol=1e-12, atol=1e-14)


# ---- C3-12: SH orthonormality ---------------------------------------------------------------------
def test_pin12_sh_orthonormal():
    nodes, wts = np.polynomial.legendre.leggauss(16)       # exact for the degree <= 6 integrands
    nphi = 32
    gram = np.zeros((16, 16))
    for ct, wt in zip(nodes, wts):
        st = math.sqrt(1 - ct * ct)
        for j in range(nphi):
            ph = 2 * math.pi * (j + 0.5) / nphi
            Y = fo.sh_basis(3, (st * math.cos(ph), st * math.sin(ph), ct)).astype(np.float64)
            gram += wt * (2 * math.pi / nphi) * np.outer(Y, Y)
    np.testing.assert_allclose(gram, np.eye(16), atol=2e-6)
    # degree-0 colour = 1/2 + c0 * sh0 ; a single higher coefficient adds Y_l(d) * value
    cam = front_camera(64, 64)
    n = 16
    mean = np.tile(np.array([[0.4, -0.3, 3.0]], np.float32), (n, 1))
    sh = np.zeros((n, 16, 3), np.float32)
    sh[:, 0, :] = 0.1
    for l in range(1, 16):
        sh[l, l, l % 3] = 0.5
    pr = fo.project(mean, np.full((n, 3), 0.1, np.float32), np.tile(np.array([[1, 0, 0, 0]], np.float32), (n, 1)),
                    np.full(n, 0.5, np.float32), sh, 3, cam35(cam), 64, 64)
    d = mean[0].astype(np.float64) - cam.cam_pos
    d = d / np.linalg.norm(d)
    Y = fo.sh_basis(3, d)
    np.testing.assert_allclose(pr["rgb"][0], 0.5 + C0 * 0.1, atol=1e-6)
    for l in range(1, 16):
        exp = np.full(3, 0.5 + C0 * 0.1)
        exp[l % 3] += Y[l] * 0.5
        np.testing.assert_allclose(pr["rgb"][l], np.maximum(exp, 0), atol=1e-6)
    # direction convention: d points from the camera to the Gaussian, Y_1 = -c1*y, Y_2 = c1*z, Y_3 = -c1*x
    Yz = fo.sh_basis(1, (0.0, 0.0, 1.0))
    np.testing.assert_allclose(Yz, [C0, 0.0, 0.4886025119029199, 0.0], atol=1e-7)
    # clamp at zero
    sh2 = np.zeros((1, 1, 3), np.float32)
    sh2[0, 0] = [-3.0, 0.0, 3.0]
    pr2 = fo.project(mean[:1], np.full((1, 3), 0.1, np.float32), np.array([[1, 0, 0, 0]], np.float32),
                     np.full(1, 0.5, np.float32), sh2, 0, cam35(cam), 64, 64)
    np.testing.assert_allclose(pr2["rgb"][0], [0.0, 0.5, 0.5 + 3 * C0], atol=1e-6)


# ---- C3-13: quaternion frames ---------------------------------------------------------------------
def test_pin13_quaternion_frames():
    np.testing.assert_allclose(fo.quat_to_rot([1, 0, 0, 0]), np.eye(3), atol=0)
    s = math.sqrt(0.5)
    R = fo.quat_to_rot([s, 0, 0, s])                                                 # 90 deg about z
    np.testing.assert_allclose(R[:, 0], [0, 1, 0], atol=1e-6)                         # t_u
    np.testing.assert_allclose(R[:, 1], [-1, 0, 0], atol=1e-6)                        # t_v
    rng = np.random.default_rng(13)
    for _ in range(200):
        q = rng.standard_normal(4) * rng.uniform(0.1, 5)          # need not be unit
        R = fo.quat_to_rot(q).astype(np.float64)
        np.testing.assert_allclose(np.cross(R[:, 0], R[:, 1]), R[:, 2], atol=2e-6)    # t_u x t_v = t_w
        np.testing.assert_allclose(R @ R.T, np.eye(3), atol=2e-6)
        v = rng.standard_normal(3)
        np.testing.assert_allclose(R @ v, _quat_rotate(q, v), atol=1e-5)


# ---- C3-14/15: instances, sort, ranges ------------------------------------------------------------
def test_pin14_splat_over_2x2_tiles():
    cam = front_camera(64, 64)
    pr = project_simple([0, 0, 4.0], [0.1, 0.1, 0.1], [1, 0, 0, 0], 0.7, [0.5, 0.5, 0.5], cam)
    b = fo.bins(pr, 64, 64, want_unsorted=True)
    assert b["M"] == 4
    assert (b["keys"] >> np.uint64(32)).tolist() == [5, 6, 9, 10]          # row-major tile ids, GW = 4
    low = (b["keys"] & np.uint64(0xFFFFFFFF)).astype(np.uint32)
    assert np.all(low == np.float32(4.0).view(np.uint32))
    assert b["ranges"][5].tolist() == [0, 1] and b["ranges"][10].tolist() == [3, 4]
    assert b["ranges"][0].tolist() == [0, 0]


def test_pin15_sort_invariants():
    cfg, sc, cam, pr = tiny_state(3)
    # force depth ties: duplicate some Gaussians' depth by copying depth values
    pr["depth"][100:200] = pr["depth"][300:400]
    b = fo.bins(pr, 64, 64, want_unsorted=True)
    M = b["M"]
    assert M == int(pr["tiles_touched"].sum()) and 1500 < M < 3000        # 2.1-2.2e3
    assert np.all(np.diff(b["offsets"].astype(np.int64)) == pr["tiles_touched"][1:])
    k, v = b["keys"], b["vals"]
    assert np.all(k[1:] >= k[:-1])
    eq = k[1:] == k[:-1]
    assert eq.sum() > 0 and np.all(v[1:][eq] > v[:-1][eq])               # stable: ties keep ascending index
    a = np.stack([b["keys_unsorted"], b["vals_unsorted"].astype(np.uint64)], 1)
    s = np.stack([k, v.astype(np.uint64)], 1)
    assert np.array_equal(a[np.lexsort((a[:, 1], a[:, 0]))], s)             # permutation of the input pairs
    # unsorted emission: Gaussian-major, tiles row-major inside the rect
    i = int(np.argmax(pr["tiles_touched"]))
    x0, y0, x1, y1 = pr["rect"][i].astype(int)
    start = int(b["offsets"][i]) - int(pr["tiles_touched"][i])
    exp_tiles = [ty * 4 + tx for ty in range(y0, y1) for tx in range(x0, x1)]
    assert (b["keys_unsorted"][start:start + len(exp_tiles)] >> np.uint64(32)).tolist() == exp_tiles
    assert np.all(b["vals_unsorted"][start:start + len(exp_tiles)] == i)
    # ranges partition [0, M)
    tiles = (k >> np.uint64(32)).astype(np.int64)
    r = b["ranges"].astype(np.int64)
    covered = 0
    for t in range(16):
        if r[t, 1] > r[t, 0]:
            assert np.all(tiles[r[t, 0]:r[t, 1]] == t)
            covered += r[t, 1] - r[t, 0]
        else:
            assert r[t].tolist() == [0, 0] and not np.any(tiles == t)
    assert covered == M


# ---- C3-16: the radius box is conservative --------------------------------------------------------
def test_pin16_conservative_box():
    cfg, sc, cam, pr = tiny_state(0, n=200)
    ys, xs = np.mgrid[0:64, 0:64]
    seen = 0
    for i in range(200):
        if pr["radius"][i] == 0:
            continue
        A, B, Cc, _ = pr["conic_opacity"][i].astype(np.float64)
        dx = pr["xy"][i, 0].astype(np.float64) - xs
        dy = pr["xy"][i, 1].astype(np.float64) - ys
        inside = (A * dx * dx + 2 * B * dx * dy + Cc * dy * dy) <= 9.0 + 1e-3
        if not inside.any():
            continue
        seen += 1
        r = float(pr["radius"][i])
        assert np.all(np.abs(dx[inside]) <= r) and np.all(np.abs(dy[inside]) <= r)
        x0, y0, x1, y1 = pr["rect"][i].astype(int)
        tx, ty = xs[inside] // 16, ys[inside] // 16
        assert np.all((tx >= x0) & (tx < x1) & (ty >= y0) & (ty < y1))
    assert seen > 100


# ---- C3-17: literal == scatter, bitwise -----------------------------------------------------------
@pytest.mark.parametrize("name,n,wh", [("tiny", None, None), ("small", 20000, 96)])
def test_pin17_literal_equals_scatter(name, n, wh):
    cfg = inputs.CONFIGS[name]
    if n:
        cfg = inputs.scaled(cfg, n=n, width=wh, height=wh)
    sc = inputs.make_scene(cfg)
    cam = inputs.make_camera(cfg, 1)
    W, H = cfg.width, cfg.height
    pr = fo.project(sc.mean, sc.scale, sc.quat, sc.opacity, sc.sh, sc.sh_degree, cam35(cam), W, H)
    order = fo.global_order(pr)
    a = fo.render_literal(pr, order, sc.feat, W, H)
    b = fo.render_scatter(pr, order, sc.feat, W, H)
    for key in ("rgb", "feat", "T", "n", "fragile"):
        assert np.array_equal(a[key], b[key]), key
    gt = inputs.make_gt_map(cfg, 1)
    n1, d1 = fo.fuse(pr, order, gt, W, H, literal=True)
    n2, d2 = fo.fuse(pr, order, gt, W, H, literal=False)
    np.testing.assert_allclose(n2, n1, rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(d2, d1, rtol=1e-11, atol=1e-13)
    # tile-binned traversal == global traversal: walking each tile's sorted range gives the same
    # visit order restricted to that tile (tiling transparency)
    b_ = fo.bins(pr, W, H)
    pos = np.empty(sc.n, np.int64)
    pos[order] = np.arange(order.shape[0])
    gw = (W + 15) // 16
    for t in (0, gw + 1, b_["ranges"].shape[0] - 1):
        s, e = b_["ranges"][t]
        assert np.all(np.diff(pos[b_["vals"][s:e]]) > 0)


# ---- C3-18: early-termination bound ---------------------------------------------------------------
def test_pin18_early_termination_bound():
    cfg = inputs.scaled(inputs.CONFIGS["small"], n=20000, width=64, height=64)
    sc = inputs.make_scene(cfg)
    cam = inputs.make_camera(cfg, 0)
    pr = fo.project(sc.mean, sc.scale, sc.quat, sc.opacity, sc.sh, sc.sh_degree, cam35(cam), 64, 64)
    order = fo.global_order(pr)
    a = fo.render_literal(pr, order, sc.feat, 64, 64)
    prm = fo.DEFAULT_PARAMS.copy()
    prm[5] = 0.0
    b = fo.render_literal(pr, order, sc.feat, 64, 64, params=prm)
    assert (a["T"] < 1e-4).mean() > 0.9                                   # the scene saturates
    assert np.all(b["n"] >= a["n"]) and np.any(b["n"] > a["n"])
    assert np.abs(a["rgb"] - b["rgb"]).max() <= 1e-4 * max(1.0, float(pr["rgb"].max()))
    assert np.abs(a["feat"] - b["feat"]).max() <= 1e-4 * float(np.abs(sc.feat).max())


# ---- C3-19: additivity / linearity ---------------------------------------------------------------
def test_pin19_fusion_additive_and_linear():
    cfg = inputs.CONFIGS["tiny"]
    sc = inputs.make_scene(cfg)
    prs, cams = [], []
    for v in (0, 1):
        cam = inputs.make_camera(cfg, v)
        prs.append(fo.project(sc.mean, sc.scale, sc.quat, sc.opacity, sc.sh, 0, cam35(cam), 64, 64))
    g0, g1 = inputs.make_gt_map(cfg, 0), inputs.make_gt_map(cfg, 1)
    nA, dA = fo.fuse(prs[0], fo.global_order(prs[0]), g0, 64, 64)
    nB, dB = fo.fuse(prs[1], fo.global_order(prs[1]), g1, 64, 64)
    nAB, dAB = fo.fuse(prs[0], fo.global_order(prs[0]), g0, 64, 64)
    nAB, dAB = fo.fuse(prs[1], fo.global_order(prs[1]), g1, 64, 64, num=nAB, den=dAB)
    np.testing.assert_allclose(nAB, nA + nB, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(dAB, dA + dB, rtol=1e-12, atol=1e-14)
    nL, _ = fo.fuse(prs[0], fo.global_order(prs[0]), 2.0 * g0 + 3.0, 64, 64)
    np.testing.assert_allclose(nL, 2.0 * nA + 3.0 * dA[:, None], rtol=1e-5, atol=1e-6)


# ---- C3-20: input-order invariance ----------------------------------------------------------------
def test_pin20_permutation_invariance():
    cfg, sc, cam, pr = tiny_state(1)
    rng = np.random.default_rng(20)
    perm = rng.permutation(sc.n)
    pr2 = fo.project(sc.mean[perm], sc.scale[perm], sc.quat[perm], sc.opacity[perm], sc.sh[perm], 0,
                     cam35(cam), 64, 64)
    assert len(np.unique(pr["depth"][pr["radius"] > 0])) == (pr["radius"] > 0).sum()    # distinct depths
    a = fo.render_literal(pr, fo.global_order(pr), sc.feat, 64, 64)
    b = fo.render_literal(pr2, fo.global_order(pr2), sc.feat[perm], 64, 64)
    for key in ("rgb", "feat", "T", "n"):
        assert np.array_equal(a[key], b[key])
    gt = inputs.make_gt_map(cfg, 1)
    n1, d1 = fo.fuse(pr, fo.global_order(pr), gt, 64, 64)
    n2, d2 = fo.fuse(pr2, fo.global_order(pr2), gt, 64, 64)
    np.testing.assert_allclose(n2, n1[perm], rtol=1e-12, atol=1e-14)
    b1, b2 = fo.bins(pr, 64, 64), fo.bins(pr2, 64, 64)
    assert np.array_equal(b1["keys"], b2["keys"]) and np.array_equal(perm[b2["vals"]], b1["vals"])


# ---- C3-21: rigid motion --------------------------------------------------------------------------
def test_pin21_rigid_motion_invariance():
    cfg, sc, cam, pr = tiny_state(0)
    rng = np.random.default_rng(21)
    qr = rng.standard_normal(4)
    Rm = np.stack([_quat_rotate(qr, e) for e in np.eye(3)], axis=1)       # columns = rotated axes
    tr = rng.uniform(-1, 1, 3)
    mean2 = (sc.mean.astype(np.float64) @ Rm.T + tr).astype(np.float32)
    qn = qr / np.linalg.norm(qr)

    def qmul(a, b):
        return np.stack([a[0]*b[:, 0] - a[1]*b[:, 1] - a[2]*b[:, 2] - a[3]*b[:, 3],
                         a[0]*b[:, 1] + a[1]*b[:, 0] + a[2]*b[:, 3] - a[3]*b[:, 2],
                         a[0]*b[:, 2] - a[1]*b[:, 3] + a[2]*b[:, 0] + a[3]*b[:, 1],
                         a[0]*b[:, 3] + a[1]*b[:, 2] - a[2]*b[:, 1] + a[3]*b[:, 0]], 1)
    quat2 = qmul(qn, sc.quat.astype(np.float64)).astype(np.float32)
    V = cam.view.astype(np.float64).reshape(4, 4)
    M = np.eye(4)
    M[:3, :3] = Rm
    M[:3, 3] = tr
    V2 = V @ np.linalg.inv(M)
    pos2 = Rm @ cam.cam_pos.astype(np.float64) + tr
    cam2 = fo.cam_array(V2.astype(np.float32), cam.proj, pos2.astype(np.float32))
    pr2 = fo.project(mean2, sc.scale, quat2, sc.opacity, sc.sh, 0, cam2, 64, 64)
    vis = (pr["radius"] > 0) & (pr2["radius"] > 0)
    assert vis.sum() > 0.95 * (pr["radius"] > 0).sum()
    np.testing.assert_allclose(pr2["xy"][vis], pr["xy"][vis], atol=2e-3)
    np.testing.assert_allclose(pr2["conic_opacity"][vis], pr["conic_opacity"][vis], rtol=2e-3, atol=1e-5)
    a = fo.render_literal(pr, fo.global_order(pr), None, 64, 64)
    b = fo.render_literal(pr2, fo.global_order(pr2), None, 64, 64)
    assert np.abs(a["rgb"] - b["rgb"]).max() < 5e-3          # fp32 projection noise moves edges slightly
    assert np.abs(a["rgb"] - b["rgb"]).mean() < 1e-5


# ---- culling rules and the Jacobian clamp (C1-P steps 1, 3, 9) ------------------------------------
def test_culling_and_clamp():
    cam = front_camera(64, 64)
    pr = project_simple([[0, 0, 0.19], [0, 0, 0.2], [0, 0, -3.0], [50.0, 0, 4.0], [np.nan, 0, 4.0]],
                        [0.01, 0.01, 0.01], [1, 0, 0, 0], 0.5, [0.5, 0.5, 0.5], cam)
    assert pr["radius"][0] == 0 and pr["tiles_touched"][0] == 0          # z < z_near
    assert pr["radius"][1] > 0                                            # z == z_near kept
    assert pr["radius"][2] == 0                                           # behind the camera
    assert pr["radius"][3] == 0 and pr["tiles_touched"][3] == 0          # far off-screen: no tile
    assert pr["radius"][4] == 0                                           # non-finite input is culled
    # clamp: at u = 3 (beyond 1.3*tan30 = 0.7506) the Jacobian uses u_c = 0.7506, not 3
    fx = 32.0 / math.tan(math.radians(30.0))
    s, z = 2.0, 2.0                 # big enough that the 3-sigma box reaches the image
    pr = project_simple([6.0, 0, z], [s, s, s], [1, 0, 0, 0], 0.5, [0.5, 0.5, 0.5], cam)
    uc = 1.3 * math.tan(math.radians(30.0))
    a = (fx * s / z) ** 2 * (1 + uc ** 2) + 0.3
    c = (fx * s / z) ** 2 + 0.3
    np.testing.assert_allclose(pr["conic_opacity"][0, :3], [1 / a, 0.0, 1 / c], rtol=1e-5, atol=1e-7)
    np.testing.assert_allclose(pr["xy"][0, 0], fx * 3.0 + 31.5, rtol=1e-6)   # the centre is NOT clamped


# ---- NEXT-4 (i): tight per-axis tile rectangles (fhgs_params.rect_mode = 1) ------------------------
def test_pin22_tight_rect_closed_form_and_conservative():
    """rect_mode 1 takes the exact bounding box of the q <= 9 ellipse: half extents 3 sqrt(Sigma_xx), 3 sqrt(Sigma_yy).
    (a) closed form on a hand-made anisotropic splat; (b) exhaustive scan: every pixel with q <= 9 lies in a tile of
    the tight rectangle, which is never larger than the radius rectangle; (c) a strongly anisotropic scene really
    shrinks; (d) everything but rect / tiles_touched is bit-identical between the two modes."""
    tight = fo.params(rect_mode=1)
    # (a) axis-aligned splat at depth 4 on the optical axis, scales (0.4, 0.05, 0.05): Sigma_xx = (fx*0.4/4)^2 + 0.3
    cam = front_camera(256, 256)
    pr = project_simple((0.0, 0.0, 4.0), (0.4, 0.05, 0.05), (1, 0, 0, 0), 0.5, (0.2, 0.4, 0.6), cam, tight)
    fx = (256 / 2) / math.tan(math.radians(30.0))
    sxx, syy = (fx * 0.4 / 4) ** 2 + 0.3, (fx * 0.05 / 4) ** 2 + 0.3
    rx, ry = math.ceil(3 * math.sqrt(sxx)), math.ceil(3 * math.sqrt(syy))
    cx = cy = 127.5
    want = [int((cx - rx) // 16), int((cy - ry) // 16), int((cx + rx) // 16) + 1, int((cy + ry) // 16) + 1]
    assert pr["rect"][0].astype(int).tolist() == want
    assert int(pr["radius"][0]) == rx                                    # the scalar radius is still ceil(3 sqrt(lambda_max))
    pr_r = project_simple((0.0, 0.0, 4.0), (0.4, 0.05, 0.05), (1, 0, 0, 0), 0.5, (0.2, 0.4, 0.6), cam)
    assert int(pr_r["tiles_touched"][0]) > int(pr["tiles_touched"][0]) > 0
    # (b), (d) random anisotropic scene
    cfg = inputs.scaled(inputs.CONFIGS["tiny"], n=300, log_scale_sigma=1.2)
    sc = inputs.make_scene(cfg)
    cam = inputs.make_camera(cfg, 1)
    args = (sc.mean, sc.scale, sc.quat, sc.opacity, sc.sh, sc.sh_degree, cam35(cam), 64, 64)
    p0, p1 = fo.project(*args), fo.project(*args, tight)
    for k in ("xy", "depth", "conic_opacity", "rgb", "radius"):
        vis = p1["radius"] > 0
        assert np.array_equal(p0[k][vis], p1[k][vis]), k
    assert np.all(p1["tiles_touched"] <= p0["tiles_touched"])
    assert p1["tiles_touched"].sum() < p0["tiles_touched"].sum()         # (c)
    ys, xs = np.mgrid[0:64, 0:64]
    seen = 0
    for i in np.nonzero(p1["radius"] > 0)[0]:
        A, B, Cc, _ = p1["conic_opacity"][i].astype(np.float64)
        dx = p1["xy"][i, 0].astype(np.float64) - xs
        dy = p1["xy"][i, 1].astype(np.float64) - ys
        inside = (A * dx * dx + 2 * B * dx * dy + Cc * dy * dy) <= 9.0 + 1e-3
        if not inside.any():
            continue
        seen += 1
        x0, y0, x1, y1 = p1["rect"][i].astype(int)
        tx, ty = xs[inside] // 16, ys[inside] // 16
        assert np.all((tx >= x0) & (tx < x1) & (ty >= y0) & (ty < y1))
    assert seen > 100


def test_pin23_tight_rect_renders_the_same_image():
    """The tile lists only serve to find the Gaussians that can reach a pixel: with either rectangle rule a tiled
    traversal (per-tile sorted ranges of fo_bins) blends exactly the fragments the tile-free literal oracle blends."""
    cfg = inputs.scaled(inputs.CONFIGS["tiny"], n=400)
    sc = inputs.make_scene(cfg)
    cam = inputs.make_camera(cfg, 2)
    for prm in (fo.DEFAULT_PARAMS, fo.params(rect_mode=1)):
        pr = fo.project(sc.mean, sc.scale, sc.quat, sc.opacity, sc.sh, sc.sh_degree, cam35(cam), 64, 64, prm)
        order = fo.global_order(pr)
        lit = fo.render_literal(pr, order, sc.feat, 64, 64)
        b = fo.bins(pr, 64, 64)
        rng = np.random.default_rng(5)
        for p in rng.integers(0, 64 * 64, size=150):
            x, y = int(p % 64), int(p // 64)
            r0, r1 = b["ranges"][(y // 16) * 4 + x // 16]
            T, n = 1.0, 0
            for g in b["vals"][int(r0):int(r1)]:
                if T < 1e-4:
                    break
                q = fo.q_value(pr["xy"][g, 0], pr["xy"][g, 1], *pr["conic_opacity"][g, :3], x, y)
                if not q <= 9.0:
                    continue
                al = min(float(np.float32(0.9999)), float(pr["conic_opacity"][g, 3]) * math.exp(-0.5 * max(float(q), 0.0)))
                T *= 1.0 - al
                n += 1
            assert n == int(lit["n"][p]) and abs(T - lit["T"][p]) < 1e-12

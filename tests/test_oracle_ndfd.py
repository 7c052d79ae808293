"""Pins for the NDFD-forward oracle (Eq. 5-6): the worked values of
SPEC.md:262-282, the O(N) == O(N^2) identity of SPEC.md:289 / PAPER.md appendix A.1, and closed forms that tie the
NDFD weights to the (already pinned) renderer.  CPU only."""
import math

import numpy as np

from oracle import fhgs_oracle as fo
from paper_2505_19154_b200 import inputs
from test_oracle_pins import manual_pr, tiny_state


def _one_pixel(ws, feats, f_gt, k=20.0, lam=0.5, mode=0, pairwise=False):
    """Fragments with blend weights `ws` (front to back) at pixel (0,0) of a 1x1 image: Gaussians centred on the
    pixel (G = 1), opacities chosen so that alpha_i T_i = ws[i]; alpha_max = 1 so that alpha = 1 is representable."""
    ws = np.asarray(ws, np.float64)
    T, ops = 1.0, []
    for w in ws:
        ops.append(w / T)
        T *= 1.0 - w / T
    n = len(ws)
    pr = manual_pr(np.zeros((n, 2)), [1.0, 0.0, 1.0], ops, [0, 0, 0], 3)
    prm = fo.DEFAULT_PARAMS.copy()
    prm[4] = 1.0   # alpha_max
    prm[5] = 0.0   # t_min: never stop (hand examples)
    order = np.arange(n, dtype=np.uint32)
    gt = np.asarray(f_gt, np.float32).reshape(1, 1, -1)
    return fo.ndfd(pr, order, np.asarray(feats, np.float32), gt, 1, 1, k=k, lam=lam, mode=mode, params=prm,
                   pairwise=pairwise)


def test_polarity_values_and_single_fragment():
    """SPEC.md:262-264 sigma(0.5) = 0.5, sigma(1) = 4.5398e-5, sigma(0) = 0.9999546 (k = 20, lambda = 0.5);
    SPEC.md:271 single fragment w = 0.6, phi = lambda -> L_gt = 0.3; N = 1 -> L_cf = 0."""
    f = [1.0, 0.0]
    for phi, sigma in [(0.5, 0.5), (1.0, 1.0 / (1.0 + math.exp(10.0))), (0.0, 1.0 / (1.0 + math.exp(-10.0)))]:
        gt = [phi, math.sqrt(1.0 - phi * phi)]
        lgt, lcf = _one_pixel([0.6], [f], gt)
        assert abs(lgt[0] - 0.6 * sigma) < 1e-7 and lcf[0] == 0.0   # opacities are stored fp32
    assert abs(1.0 / (1.0 + math.exp(10.0)) - 4.5398e-5) < 1e-9 and abs(1.0 / (1.0 + math.exp(-10.0)) - 0.9999546) < 1e-7
    lgt, _ = _one_pixel([0.6], [f], [0.5, math.sqrt(0.75)])
    assert abs(lgt[0] - 0.3) < 1e-7
    lgt, lcf = _one_pixel([], np.zeros((0, 2)), [1.0, 0.0])   # empty pixel
    assert lgt[0] == 0.0 and lcf[0] == 0.0


def test_two_fragments_hand_values():
    """two fragments, orthogonal unit features, w1 = w2 = 0.5, sigma_2 = 1 -> L_cf = 0.25;
    identical features -> L_cf = 0."""
    f1, f2 = [1.0, 0.0], [0.0, 1.0]
    lgt, lcf = _one_pixel([0.5, 0.5], [f1, f2], [0.0, -1.0])       # phi_2 = -1 -> sigma_2 = 1 - 9e-14
    assert abs(lcf[0] - 0.25) < 1e-7
    s1 = 1.0 / (1.0 + math.exp(20.0 * (0.0 - 0.5)))
    assert abs(lgt[0] - (0.5 * s1 + 0.5)) < 1e-7
    # far -> near accumulation: the partner set flips, sigma_1 multiplies the pair instead of sigma_2
    _, lcf_r = _one_pixel([0.5, 0.5], [f1, f2], [0.0, -1.0], mode=1)
    assert abs(lcf_r[0] - s1 * 0.25) < 1e-7
    _, lcf_same = _one_pixel([0.5, 0.3], [f1, f1], [0.6, 0.8])
    assert abs(lcf_same[0]) < 1e-12


def test_recurrence_equals_pairwise_sum():
    """The O(N) cumulative form of Eq. 6 equals the explicit double sum, both
    accumulation orders, on the Tiny scene with unit features and a random unit-norm map."""
    cfg, sc, cam, pr = tiny_state(1)
    order = fo.global_order(pr)
    rng = np.random.default_rng(5)
    feat = rng.standard_normal((sc.n, 12)).astype(np.float32)
    feat /= np.linalg.norm(feat, axis=1, keepdims=True)
    gt = rng.standard_normal((cfg.height, cfg.width, 12)).astype(np.float32)
    gt /= np.linalg.norm(gt, axis=2, keepdims=True)
    for mode in (0, 1):
        lgt, lcf, pw = fo.ndfd(pr, order, feat, gt, cfg.width, cfg.height, mode=mode, pairwise=True)
        assert np.abs(lcf).max() > 1e-3
        np.testing.assert_allclose(lcf, pw, rtol=1e-10, atol=1e-14)


def test_constant_polarity_ties_ndfd_to_the_renderer():
    """k = 0 makes sigma = 1/2 for every fragment.  Then L_gt = (1 - T_final)/2, and for unit features
    L_cf = ((1 - T_final)^2 - |feat_img|^2 - sum_i w_i^2 (1 - 1)) / 4 = ((sum w)^2 - |F_N|^2) / 4 in either accumulation
    order: both are functions of the renderer's outputs (pinned by C3-3/6/7), so the NDFD traversal uses exactly the
    renderer's weights, cut-off and stopping rule."""
    cfg, sc, cam, pr = tiny_state(0)
    order = fo.global_order(pr)
    rng = np.random.default_rng(9)
    feat = rng.standard_normal((sc.n, 8)).astype(np.float32)
    feat /= np.linalg.norm(feat, axis=1, keepdims=True)
    gt = rng.standard_normal((cfg.height, cfg.width, 8)).astype(np.float32)
    r = fo.render_literal(pr, order, feat, cfg.width, cfg.height)
    W = 1.0 - r["T"]
    for mode in (0, 1):
        lgt, lcf = fo.ndfd(pr, order, feat, gt, cfg.width, cfg.height, k=0.0, mode=mode)
        np.testing.assert_allclose(lgt, 0.5 * W, atol=1e-12)
        # sum_{j<i} w_i w_j (1 - f_i.f_j) = ((sum w)^2 - sum w_i^2)/2 - (|F|^2 - sum w_i^2 |f_i|^2)/2; |f_i| = 1 up to fp32
        np.testing.assert_allclose(lcf, 0.25 * (W * W - (r["feat"] ** 2).sum(axis=1)), atol=2e-7)
    assert W.max() > 0.5


def test_bounds_and_monotonicity():
    """0 <= L_gt <= sum w <= 1; L_cf >= 0 for unit features (1 - f_i.f_j >= 0); raising lambda raises every sigma,
    hence L_gt."""
    cfg, sc, cam, pr = tiny_state(2)
    order = fo.global_order(pr)
    rng = np.random.default_rng(11)
    feat = rng.standard_normal((sc.n, 16)).astype(np.float32)
    feat /= np.linalg.norm(feat, axis=1, keepdims=True)
    gt = rng.standard_normal((cfg.height, cfg.width, 16)).astype(np.float32)
    gt /= np.linalg.norm(gt, axis=2, keepdims=True)
    r = fo.render_literal(pr, order, None, cfg.width, cfg.height)
    lgt, lcf = fo.ndfd(pr, order, feat, gt, cfg.width, cfg.height)
    assert np.all(lgt >= 0) and np.all(lgt <= 1.0 - r["T"] + 1e-12) and np.all(lcf >= -1e-9)
    lgt2, _ = fo.ndfd(pr, order, feat, gt, cfg.width, cfg.height, lam=0.7)
    assert np.all(lgt2 >= lgt - 1e-15) and (lgt2 - lgt).max() > 1e-3


# ---- NEXT-2: backward at the w level -------------------------------------------------------------
def _one_pixel_backward(ws, feats, f_gt, lam1, lam2, k=20.0, lam=0.5):
    ws = np.asarray(ws, np.float64)
    T, ops = 1.0, []
    for w in ws:
        ops.append(w / T)
        T *= 1.0 - w / T
    n = len(ws)
    pr = manual_pr(np.zeros((n, 2)), [1.0, 0.0, 1.0], ops, [0, 0, 0], 3)
    prm = fo.DEFAULT_PARAMS.copy()
    prm[4] = 1.0 + 1e-3   # alpha_max above 1: nothing is clamped in the hand examples
    prm[5] = 0.0
    gt = np.asarray(f_gt, np.float32).reshape(1, 1, -1)
    return fo.ndfd_backward(pr, np.arange(n, dtype=np.uint32), np.asarray(feats, np.float32), gt, 1, 1, k=k, lam=lam,
                            lam1=lam1, lam2=lam2, params=prm), np.asarray(ops)


def test_backward_hand_values():
    """SPEC.md:343 dL_gt/dw = sigma; SPEC.md:354 the two-orthogonal-fragment example: dL_cf/dw_1 = sigma_2 w_2 = 0.5,
    dL_cf/dw_2 = sigma_2 (W_1 - F_1.f_2) = 0.5; SPEC.md:363 dL/dalpha_near = dL/dw_near - dL/dw_far w_far / (1 - alpha_near).
    The Gaussians sit on the pixel (G = 1), so dL/dop = dL/dalpha."""
    # single fragment, L_gt only: dL/dop = T_1 sigma = sigma
    (L, g), _ = _one_pixel_backward([0.6], [[1.0, 0.0]], [0.5, math.sqrt(0.75)], 1.0, 0.0)
    assert abs(L - 0.3) < 1e-7 and abs(g[0] - 0.5) < 1e-7
    # two orthogonal fragments, L_cf only, w = (0.5, 0.25): alpha = (0.5, 0.5), T = (1, 0.5), sigma_2 ~ 1
    (L, g), ops = _one_pixel_backward([0.5, 0.25], [[1.0, 0.0], [0.0, 1.0]], [0.0, -1.0], 0.0, 1.0)
    assert abs(L - 0.125) < 1e-7                         # sigma_2 w_2 (W_1 - F_1.f_2) = 0.25 * 0.5
    gw1, gw2 = 0.25, 0.5                                 # sigma_2 w_2 (1 - 0);  sigma_2 (W_1 - 0)   (SPEC.md:354 pattern)
    da2 = 0.5 * gw2                                      # far fragment: T_2 dL/dw_2
    da1 = 1.0 * gw1 - gw2 * 0.25 / (1.0 - 0.5)           # near fragment: SPEC.md:363
    np.testing.assert_allclose(g, [da1, da2], atol=1e-7)
    assert abs(g[0]) < 1e-7      # L_cf = a1 (1 - a1) a2: d/da1 vanishes at a1 = 1/2; d/da2 = a1 (1 - a1) = 1/4


def test_backward_loss_matches_forward_and_finite_differences():
    """L equals the forward oracle's sum; dL/d opacity matches central finite differences of the FORWARD oracle
     on the Tiny scene (t_min = 0 so that the fragment lists do not change)."""
    cfg, sc, cam, pr = tiny_state(3)
    order = fo.global_order(pr)
    rng = np.random.default_rng(21)
    feat = rng.standard_normal((sc.n, 12)).astype(np.float32)
    feat /= np.linalg.norm(feat, axis=1, keepdims=True)
    gt = rng.standard_normal((cfg.height, cfg.width, 12)).astype(np.float32)
    gt /= np.linalg.norm(gt, axis=2, keepdims=True)
    prm = fo.DEFAULT_PARAMS.copy()
    prm[5] = 0.0
    lam1, lam2 = 0.7, 1.3
    L, grad = fo.ndfd_backward(pr, order, feat, gt, cfg.width, cfg.height, lam1=lam1, lam2=lam2, params=prm)

    def forward_total(p):
        lgt, lcf = fo.ndfd(p, order, feat, gt, cfg.width, cfg.height, params=prm)
        return lam1 * lgt.sum() + lam2 * lcf.sum()

    assert abs(L - forward_total(pr)) <= 1e-9 * abs(L)
    probe = np.argsort(-np.abs(grad))[[0, 1, 2, 5, 10, 50, 200]]
    assert np.abs(grad[probe]).min() > 0
    for g in probe:
        o0 = pr["conic_opacity"][g, 3]
        hi, lo = np.float32(o0 * (1 + 2e-3)), np.float32(o0 * (1 - 2e-3))
        p_hi = dict(pr, conic_opacity=pr["conic_opacity"].copy()); p_hi["conic_opacity"][g, 3] = hi
        p_lo = dict(pr, conic_opacity=pr["conic_opacity"].copy()); p_lo["conic_opacity"][g, 3] = lo
        fd = (forward_total(p_hi) - forward_total(p_lo)) / (float(hi) - float(lo))
        assert abs(fd - grad[g]) <= 2e-4 * max(abs(grad[g]), 1e-3), (g, fd, grad[g])


def test_backward_linearity_and_clamp():
    """dL/dop is linear in (lam1, lam2); a fragment clamped at alpha_max passes no gradient to its opacity."""
    cfg, sc, cam, pr = tiny_state(0)
    order = fo.global_order(pr)
    rng = np.random.default_rng(22)
    feat = rng.standard_normal((sc.n, 8)).astype(np.float32)
    feat /= np.linalg.norm(feat, axis=1, keepdims=True)
    gt = rng.standard_normal((cfg.height, cfg.width, 8)).astype(np.float32)
    gt /= np.linalg.norm(gt, axis=2, keepdims=True)
    _, g10 = fo.ndfd_backward(pr, order, feat, gt, cfg.width, cfg.height, lam1=1.0, lam2=0.0)
    _, g01 = fo.ndfd_backward(pr, order, feat, gt, cfg.width, cfg.height, lam1=0.0, lam2=1.0)
    _, g23 = fo.ndfd_backward(pr, order, feat, gt, cfg.width, cfg.height, lam1=2.0, lam2=3.0)
    np.testing.assert_allclose(g23, 2.0 * g10 + 3.0 * g01, rtol=1e-10, atol=1e-12)
    # one opaque Gaussian on a pixel centre: op * G = 1 > alpha_max -> clamped there; only off-centre pixels pass gradient
    prm = fo.DEFAULT_PARAMS.copy()
    p1 = manual_pr([[0.0, 0.0]], [1.0, 0.0, 1.0], [1.0], [0, 0, 0], 3)
    gt1 = np.zeros((1, 1, 2), np.float32); gt1[..., 0] = 1.0
    _, gc = fo.ndfd_backward(p1, np.array([0], np.uint32), np.array([[0.0, 1.0]], np.float32), gt1, 1, 1, lam1=1.0, lam2=0.0,
                             params=prm)
    assert gc[0] == 0.0

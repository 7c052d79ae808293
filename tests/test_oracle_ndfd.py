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

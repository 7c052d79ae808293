"""Oracle pins against the worked values the reference texts print (tests/golden/spec_worked_values.json;
every entry carries its SPEC.md / PAPER.md citation).  CPU only."""
import json
import os

import numpy as np

from oracle import fhgs_oracle as fo

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "spec_worked_values.json")))
W = H = 32


def _state(xy, conic, op, rgb):
    """Hand-made projected state (step P outputs) so that compositing is pinned independently of projection."""
    n = len(op)
    return dict(xy=np.asarray(xy, np.float32).reshape(n, 2), depth=np.arange(1, n + 1, dtype=np.float32),
                conic_opacity=np.concatenate([np.asarray(conic, np.float32).reshape(n, 3),
                                              np.asarray(op, np.float32).reshape(n, 1)], axis=1),
                rgb=np.asarray(rgb, np.float32).reshape(n, 3), radius=np.full(n, 64, np.int32),
                rect=np.tile(np.array([0, 0, 2, 2], np.uint16), (n, 1)), tiles_touched=np.full(n, 4, np.uint32))


def _render_at(pr, x, y, feat=None):
    order = fo.global_order(pr)
    return fo.render_literal(pr, order, feat, W, H, pix=np.array([y * W + x], np.int32))


def test_gaussian_density_values():
    g = GOLD["gaussian_density"]
    for c in g["cases"]:
        # a unit-covariance splat centred on pixel (10,10), opacity 1: alpha at (10+u, 10+v) is G(u,v)
        pr = _state([[10.0, 10.0]], [[1.0, 0.0, 1.0]], [1.0], [[1.0, 1.0, 1.0]])
        o = _render_at(pr, 10 + int(c["u"]), 10 + int(c["v"]))
        got = 1.0 - o["T"][0] if c["G"] < 1.0 else o["rgb"][0, 0] / 0.9999 * 1.0
        want = c["G"] if c["G"] < 1.0 else 1.0
        if c["G"] == 1.0:   # alpha is clamped to alpha_max = 0.9999: G = 1 -> w = 0.9999
            assert abs(o["rgb"][0, 0] - 0.9999) < 1e-6
        else:
            assert abs(got - want) < g["abs_tol"], (c, got)


def test_two_fragment_blend():
    g = GOLD["two_fragment_blend"]
    # very wide splats (conic ~ 0) so that G = 1 at the pixel and alpha = opacity
    pr = _state([[5.0, 5.0], [5.0, 5.0]], [[0.0, 0.0, 0.0]] * 2, g["alpha"], g["colour"])
    feat = np.eye(2, dtype=np.float32)          # feature channel i carries w_i
    o = _render_at(pr, 5, 5, feat)
    assert np.allclose(o["rgb"][0], g["out_colour"], atol=1e-12)
    assert np.allclose(o["feat"][0], g["w"], atol=1e-12)
    assert abs((1.0 - o["T"][0]) - g["weight_sum"]) < 1e-12 and o["n"][0] == 2
    # fusion sees the same weights: den_i = w_i for a single pixel... over the whole image it is w_i per pixel
    gt = np.ones((H, W, 1), np.float32)
    num, den = fo.fuse(pr, fo.global_order(pr), gt, W, H, literal=True)
    assert np.allclose(den, np.array(g["w"]) * W * H, rtol=1e-12)


def test_opaque_fragment_and_empty_list():
    g = GOLD["opaque_fragment"]
    pr = _state([[5.0, 5.0]], [[0.0, 0.0, 0.0]], [1.0], [g["colour"]])   # op*G = 1 -> clamped to alpha_max
    o = _render_at(pr, 5, 5)
    assert np.allclose(o["rgb"][0], g["out_colour"], atol=g["abs_tol"])
    assert abs((1.0 - o["T"][0]) - g["weight_sum"]) < g["abs_tol"]
    e = GOLD["empty_list"]
    pr0 = _state(np.zeros((0, 2)), np.zeros((0, 3)), np.zeros(0), np.zeros((0, 3)))
    o = fo.render_literal(pr0, np.zeros(0, np.uint32), None, W, H, pix=np.array([0], np.int32))
    assert np.allclose(o["rgb"][0], e["out_colour"]) and 1.0 - o["T"][0] == e["weight_sum"]


def test_quaternion_frames():
    g = GOLD["quaternion_frames"]
    for c in g["cases"]:
        R = fo.quat_to_rot(np.array(c["q_wxyz"], np.float32))
        for col, name in enumerate(("t_u", "t_v", "t_w")):
            assert np.abs(R[:, col] - np.array(c[name], np.float32)).max() < g["abs_tol"], (c, name)


def test_2x2_tile_block_instances():
    g = GOLD["tile_block_2x2"]
    pr = _state([[15.5, 15.5]], [[1.0, 0.0, 1.0]], [0.5], [[1, 1, 1]])
    pr["depth"][:] = 2.5
    b = fo.bins(pr, W, H)
    assert b["M"] == g["instances"]
    assert len(set((b["keys"] & np.uint64(0xffffffff)).tolist())) == 1      # identical depth keys
    assert sorted((b["keys"] >> np.uint64(32)).tolist()) == [0, 1, 2, 3]


def test_unit_feature_splat_centre_pixel():
    pr = _state([[16.0, 16.0]], [[0.05, 0.0, 0.05]], [0.7], [[1, 1, 1]])
    feat = np.zeros((1, 4), np.float32); feat[0, 0] = 1.0                  # f = e0
    o = _render_at(pr, 16, 16, feat)
    w = 1.0 - o["T"][0]
    assert abs(w - 0.7) < 1e-7 and abs(o["feat"][0, 0] - w) < 1e-12 and np.all(o["feat"][0, 1:] == 0)

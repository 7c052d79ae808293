"""ctypes loader for the CPU oracle (oracle/fhgs_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this module.  It never imports the CUDA package and shares no code with it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fhgs_oracle.c")
_LIB = os.path.join(_HERE, "libfhgs_oracle.so")

DEFAULT_PARAMS = np.array([0.2, 0.3, 1.3, 9.0, 0.9999, 1e-4, 1e-8, 0.0, 0.0, 0.0, 0.0, 0.0], dtype=np.float32)
# order: z_near, cov_dilation, jac_clamp, q_cutoff, alpha_max, t_min, den_eps, bg[3],
#        rect_mode (0 scalar radius | 1 tight per-axis extents), primitive (0 EWA Gaussian | 1 surfel)
P_RECT, P_PRIM = 10, 11


def params(**kw) -> np.ndarray:
    """DEFAULT_PARAMS with overrides by name (rect_mode=1, primitive=1, bg=(r,g,b), ...)."""
    names = ["z_near", "cov_dilation", "jac_clamp", "q_cutoff", "alpha_max", "t_min", "den_eps"]
    p = DEFAULT_PARAMS.copy()
    for k, v in kw.items():
        if k == "bg":
            p[7:10] = v
        elif k == "rect_mode":
            p[P_RECT] = v
        elif k == "primitive":
            p[P_PRIM] = v
        else:
            p[names.index(k)] = v
    return p


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               _SRC, "-o", _LIB, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.fo_count_instances.restype = C.c_uint64
        _lib.fo_bins.restype = C.c_uint64
        _lib.fo_global_order.restype = C.c_int
        _lib.fo_num_threads.restype = C.c_int
        _lib.fo_q.restype = C.c_float
        _lib.fo_q.argtypes = [C.c_float] * 5 + [C.c_int, C.c_int]
    return _lib


def num_threads() -> int:
    return int(lib().fo_num_threads())


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def cam_array(view, proj, cam_pos) -> np.ndarray:
    return np.concatenate([_f32(view).ravel(), _f32(proj).ravel(), _f32(cam_pos).ravel()])


def sh_basis(degree: int, d) -> np.ndarray:
    out = np.zeros((degree + 1) ** 2, dtype=np.float32)
    lib().fo_sh_basis(C.c_int(degree), C.c_float(d[0]), C.c_float(d[1]), C.c_float(d[2]), _p(out))
    return out


def quat_to_rot(q) -> np.ndarray:
    q = _f32(q)
    out = np.zeros(9, dtype=np.float32)
    lib().fo_quat_to_rot(_p(q), _p(out))
    return out.reshape(3, 3)


def q_value(pxg, pyg, A, B, Cc, x, y) -> float:
    return float(lib().fo_q(pxg, pyg, A, B, Cc, int(x), int(y)))


def project(mean, scale, quat, opacity, sh, sh_degree, cam, W, H, params=DEFAULT_PARAMS):
    """Step P.  Returns dict of xy, depth, conic_opacity, rgb, radius, rect, tiles_touched."""
    mean, scale, quat, opacity, sh = map(_f32, (mean, scale, quat, opacity, sh))
    n = mean.shape[0]
    out = dict(xy=np.zeros((n, 2), np.float32), depth=np.zeros(n, np.float32),
               conic_opacity=np.zeros((n, 4), np.float32), rgb=np.zeros((n, 3), np.float32),
               radius=np.zeros(n, np.int32), rect=np.zeros((n, 4), np.uint16),
               tiles_touched=np.zeros(n, np.uint32))
    common = (C.c_int(n), C.c_int(sh_degree), _p(mean), _p(scale), _p(quat), _p(opacity),
              _p(sh), _p(_f32(cam)), C.c_int(W), C.c_int(H), _p(_f32(params)),
              _p(out["xy"]), _p(out["depth"]), _p(out["conic_opacity"]), _p(out["rgb"]),
              _p(out["radius"]), _p(out["rect"]), _p(out["tiles_touched"]))
    if float(params[P_PRIM]) != 0.0:      # NEXT-3: 2-D surfels; the projected state carries the per-splat ray transform
        out["ray_transform"] = np.zeros((n, 12), np.float32)
        lib().fo_project_surfel(*common, _p(out["ray_transform"]))
    else:
        lib().fo_project(*common)
    return out


class _surfel:
    """Selects the surfel evaluation (fo_set_surfel) for the duration of one oracle call when the projected state
    `pr` came from the surfel projection."""

    def __init__(self, pr):
        self.rt = pr.get("ray_transform")

    def __enter__(self):
        if self.rt is not None:
            lib().fo_set_surfel(_p(np.ascontiguousarray(self.rt)))

    def __exit__(self, *a):
        if self.rt is not None:
            lib().fo_set_surfel(None)


def surfel_terms(rt_row, x, y):
    """(p[3], num, den) of fo_surfel_terms for one surfel and pixel: (u, v) = p[:2] / p[2], q = num / den."""
    rt_row = _f32(rt_row)
    p3 = np.zeros(3, np.float32)
    num, den = C.c_float(0), C.c_float(0)
    lib().fo_surfel_terms(_p(rt_row), C.c_int(int(x)), C.c_int(int(y)), _p(p3), C.byref(num), C.byref(den))
    return p3, float(num.value), float(den.value)


def bins(pr, W, H, want_unsorted=False):
    """Step S.  Returns dict M, offsets, keys, vals, ranges (+ keys_unsorted, vals_unsorted)."""
    n = pr["radius"].shape[0]
    tt = np.ascontiguousarray(pr["tiles_touched"])
    m = int(lib().fo_count_instances(C.c_int(n), _p(tt)))
    gw, gh = (W + 15) // 16, (H + 15) // 16
    out = dict(M=m, offsets=np.zeros(n, np.uint32), keys=np.zeros(m, np.uint64),
               vals=np.zeros(m, np.uint32), ranges=np.zeros((gw * gh, 2), np.uint32))
    ku = np.zeros(m, np.uint64) if want_unsorted else None
    vu = np.zeros(m, np.uint32) if want_unsorted else None
    m2 = lib().fo_bins(C.c_int(n), _p(tt), _p(np.ascontiguousarray(pr["rect"])),
                       _p(np.ascontiguousarray(pr["depth"])), C.c_int(W), C.c_int(H),
                       _p(out["offsets"]), _p(ku), _p(vu), _p(out["keys"]), _p(out["vals"]),
                       _p(out["ranges"]))
    assert int(m2) == m
    if want_unsorted:
        out["keys_unsorted"], out["vals_unsorted"] = ku, vu
    return out


def global_order(pr) -> np.ndarray:
    n = pr["radius"].shape[0]
    order = np.zeros(max(n, 1), np.uint32)
    c = lib().fo_global_order(C.c_int(n), _p(np.ascontiguousarray(pr["radius"])),
                              _p(np.ascontiguousarray(pr["depth"])), _p(order))
    return order[:c].copy()


def _render_out(npix, D, want_feat):
    return dict(rgb=np.zeros((npix, 3), np.float64),
                feat=np.zeros((npix, D), np.float64) if want_feat else None,
                T=np.zeros(npix, np.float64), n=np.zeros(npix, np.uint32),
                fragile=np.zeros(npix, np.uint8))


def render_literal(pr, order, feat, W, H, params=DEFAULT_PARAMS, pix=None):
    """Step R, literal per-pixel walk over all visible Gaussians.  `pix`: optional int32 array of
    linear pixel ids (y*W+x); default = the whole image."""
    feat32 = None if feat is None else _f32(feat)
    D = 0 if feat32 is None else feat32.shape[1]
    if pix is not None:
        pix = np.ascontiguousarray(pix, dtype=np.int32)
    npix = W * H if pix is None else pix.shape[0]
    o = _render_out(npix, D, feat32 is not None)
    with _surfel(pr):
      lib().fo_render_literal(C.c_int(order.shape[0]), _p(order), C.c_int(D), _p(pr["xy"]),
                            _p(pr["conic_opacity"]), _p(pr["rgb"]), _p(feat32), C.c_int(W),
                            C.c_int(H), _p(_f32(params)), C.c_int64(npix), _p(pix), _p(o["rgb"]),
                            _p(o["feat"]), _p(o["T"]), _p(o["n"]), _p(o["fragile"]))
    return o


def render_scatter(pr, order, feat, W, H, params=DEFAULT_PARAMS):
    feat32 = None if feat is None else _f32(feat)
    D = 0 if feat32 is None else feat32.shape[1]
    o = _render_out(W * H, D, feat32 is not None)
    with _surfel(pr):
      lib().fo_render_scatter(C.c_int(order.shape[0]), _p(order), C.c_int(D), _p(pr["xy"]),
                            _p(pr["conic_opacity"]), _p(pr["rgb"]), _p(feat32), _p(pr["radius"]),
                            C.c_int(W), C.c_int(H), _p(_f32(params)), _p(o["rgb"]), _p(o["feat"]),
                            _p(o["T"]), _p(o["n"]), _p(o["fragile"]))
    return o


def fuse(pr, order, gt, W, H, params=DEFAULT_PARAMS, num=None, den=None, literal=False):
    """Step F.  Accumulates into (num, den) (created zero if None) and returns them."""
    gt32 = _f32(gt)
    D = gt32.shape[-1]
    n = pr["radius"].shape[0]
    if num is None:
        num = np.zeros((n, D), np.float64)
        den = np.zeros(n, np.float64)
    if literal:
      with _surfel(pr):
        lib().fo_fuse_literal(C.c_int(n), C.c_int(order.shape[0]), _p(order), C.c_int(D),
                              _p(pr["xy"]), _p(pr["conic_opacity"]), _p(gt32), C.c_int(W),
                              C.c_int(H), _p(_f32(params)), _p(num), _p(den))
    else:
      with _surfel(pr):
        lib().fo_fuse_scatter(C.c_int(n), C.c_int(order.shape[0]), _p(order), C.c_int(D),
                              _p(pr["xy"]), _p(pr["conic_opacity"]), _p(pr["radius"]), _p(gt32),
                              C.c_int(W), C.c_int(H), _p(_f32(params)), _p(num), _p(den))
    return num, den


def finalize(num, den, feat_prev, den_eps=1e-8, l2norm=False) -> np.ndarray:
    n, D = num.shape
    out = np.ascontiguousarray(feat_prev, dtype=np.float64).copy()
    lib().fo_fuse_finalize(C.c_int(n), C.c_int(D), _p(num), _p(den), C.c_double(den_eps),
                           C.c_int(1 if l2norm else 0), _p(out))
    return out


def ndfd(pr, order, feat, gt, W, H, k=20.0, lam=0.5, mode=0, params=DEFAULT_PARAMS, pix=None, pairwise=False):
    """NDFD forward: per-pixel L_gt, L_cf (float64) over `pix` (int32 linear ids; None = all).
    mode 0: W, F accumulated in blend order (front to back); mode 1: from far to near.  pairwise=True also returns
    the explicit O(N^2) double sum of Eq. 6 (third array)."""
    feat32, gt32 = _f32(feat), _f32(gt)
    D = feat32.shape[1]
    if pix is not None:
        pix = np.ascontiguousarray(pix, dtype=np.int32)
    npix = W * H if pix is None else pix.shape[0]
    lgt, lcf = np.zeros(npix, np.float64), np.zeros(npix, np.float64)
    args = (C.c_int(order.shape[0]), _p(order), C.c_int(D), _p(pr["xy"]), _p(pr["conic_opacity"]), _p(feat32), _p(gt32),
            C.c_int(W), C.c_int(H), _p(_f32(params)), C.c_double(k), C.c_double(lam), C.c_int(mode), C.c_int64(npix), _p(pix))
    with _surfel(pr):
        lib().fo_ndfd_literal(*args, _p(lgt), _p(lcf))
    if not pairwise:
        return lgt, lcf
    pw = np.zeros(npix, np.float64)
    with _surfel(pr):
        lib().fo_ndfd_pairwise(*args, _p(pw))
    return lgt, lcf, pw


def ndfd_backward(pr, order, feat, gt, W, H, k=20.0, lam=0.5, lam1=1.0, lam2=1.0, params=DEFAULT_PARAMS, pix=None):
    """NDFD backward at the w level: returns (L, grad_opacity[n]) with
    L = sum over `pix` of lam1 L_gt + lam2 L_cf (blend-order accumulation) and grad_opacity = dL/d opacity."""
    feat32, gt32 = _f32(feat), _f32(gt)
    D = feat32.shape[1]
    n = pr["radius"].shape[0]
    if pix is not None:
        pix = np.ascontiguousarray(pix, dtype=np.int32)
    npix = W * H if pix is None else pix.shape[0]
    grad = np.zeros(n, np.float64)
    fn = lib().fo_ndfd_backward
    fn.restype = C.c_double
    with _surfel(pr):
        L = fn(C.c_int(order.shape[0]), _p(order), C.c_int(D), _p(pr["xy"]), _p(pr["conic_opacity"]), _p(feat32), _p(gt32),
               C.c_int(W), C.c_int(H), _p(_f32(params)), C.c_double(k), C.c_double(lam), C.c_double(lam1), C.c_double(lam2),
               C.c_int64(npix), _p(pix), _p(grad))
    return float(L), grad

"""Thin ctypes binding of libfhgs.so (include/fhgs.h).  Argument marshalling only: every step of
the path runs in the CUDA kernels.  torch supplies device memory and the stream.

The library is loaded on import of this module and import FAILS LOUDLY if it is missing or cannot
be loaded: there is no CPU fallback (and this module never imports oracle/)."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("FHGS_LIB") or os.path.join(_HERE, "libfhgs.so")   # FHGS_LIB: load another build of the same ABI

FHGS_OK, FHGS_ERR_INTERNAL, FHGS_ERR_INVALID, FHGS_ERR_CAPACITY = 0, 1, 2, 3
FHGS_F32, FHGS_F16, FHGS_BF16 = 0, 1, 2
FHGS_SORT_FULL_KEY = 1
FHGS_FUSE_ZERO, FHGS_FUSE_FINALIZE, FHGS_FUSE_L2NORM, FHGS_FUSE_FINALIZE_ONLY, FHGS_FUSE_ZERO_ONLY = 1, 2, 4, 8, 16
FHGS_FUSE_ZERO_TOUCHED = 32
FHGS_RECT_RADIUS, FHGS_RECT_TIGHT = 0, 1
FHGS_PRIM_EWA, FHGS_PRIM_SURFEL = 0, 1
FHGS_NDFD_BLEND_ORDER, FHGS_NDFD_FAR_TO_NEAR = 0, 1

EXPORTS = ["fhgs_create", "fhgs_destroy", "fhgs_last_error", "fhgs_version", "fhgs_default_params",
           "fhgs_scratch_bytes", "fhgs_scratch_tile_visited", "fhgs_set_diagnostics", "fhgs_project", "fhgs_bin_sort", "fhgs_render", "fhgs_fuse_features", "fhgs_ndfd_forward", "fhgs_ndfd_backward_work_bytes", "fhgs_ndfd_backward",
           "fhgs_frame_host", "fhgs_ffma_peak", "fhgs_scan_offsets_static_max_n", "fhgs_scan_offsets_static", "fhgs_render_fuse"]


class FhgsError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__(f"fhgs status {status}: {text}")
        self.status = status


class CGaussians(C.Structure):
    _fields_ = [("n", C.c_int32), ("sh_degree", C.c_int32), ("feat_dim", C.c_int32), ("feat_dtype", C.c_int32),
                ("mean", C.c_void_p), ("scale", C.c_void_p), ("quat", C.c_void_p), ("opacity", C.c_void_p),
                ("sh", C.c_void_p), ("feat", C.c_void_p)]


class CCamera(C.Structure):
    _fields_ = [("view", C.c_float * 16), ("proj", C.c_float * 16), ("cam_pos", C.c_float * 3),
                ("width", C.c_int32), ("height", C.c_int32)]


class CParams(C.Structure):
    _fields_ = [("z_near", C.c_float), ("cov_dilation", C.c_float), ("jac_clamp", C.c_float),
                ("q_cutoff", C.c_float), ("alpha_max", C.c_float), ("t_min", C.c_float),
                ("den_eps", C.c_float), ("bg", C.c_float * 3), ("rect_mode", C.c_int32), ("primitive", C.c_int32)]


class CViewState(C.Structure):
    _fields_ = [("n", C.c_int32), ("width", C.c_int32), ("height", C.c_int32), ("sorted_buf", C.c_int32),
                ("capacity", C.c_uint64),
                ("xy", C.c_void_p), ("depth", C.c_void_p), ("conic_opacity", C.c_void_p), ("rgb", C.c_void_p),
                ("radius", C.c_void_p), ("rect", C.c_void_p), ("tiles_touched", C.c_void_p),
                ("offsets", C.c_void_p), ("num_instances", C.c_void_p),
                ("keys", C.c_void_p * 2), ("vals", C.c_void_p * 2), ("ranges", C.c_void_p),
                ("scratch", C.c_void_p), ("scratch_bytes", C.c_size_t), ("ray_transform", C.c_void_p)]


class CHostFrame(C.Structure):
    _fields_ = [("mean", C.c_void_p), ("scale", C.c_void_p), ("quat", C.c_void_p), ("opacity", C.c_void_p),
                ("sh", C.c_void_p), ("feat", C.c_void_p), ("gt", C.c_void_p), ("out_rgb", C.c_void_p),
                ("out_feat", C.c_void_p), ("fused_feat", C.c_void_p)]


class CFrameWorkspace(C.Structure):
    _fields_ = [("out_rgb", C.c_void_p), ("out_feat", C.c_void_p), ("gt", C.c_void_p), ("num", C.c_void_p),
                ("den", C.c_void_p), ("fused_feat", C.c_void_p)]


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2505_19154_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp = C.c_void_p
    lib.fhgs_version.restype = C.c_char_p
    lib.fhgs_last_error.restype = C.c_char_p
    lib.fhgs_last_error.argtypes = [vp]
    lib.fhgs_create.argtypes = [C.POINTER(vp), C.c_int]
    lib.fhgs_destroy.argtypes = [vp]
    lib.fhgs_destroy.restype = None
    lib.fhgs_default_params.argtypes = [C.POINTER(CParams)]
    lib.fhgs_default_params.restype = None
    lib.fhgs_scratch_bytes.restype = C.c_size_t
    lib.fhgs_scratch_bytes.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_uint64]
    lib.fhgs_scratch_tile_visited.restype = C.c_size_t
    lib.fhgs_scratch_tile_visited.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_uint64]
    lib.fhgs_set_diagnostics.restype = None
    lib.fhgs_set_diagnostics.argtypes = [vp, C.c_int]
    lib.fhgs_project.argtypes = [vp, C.POINTER(CGaussians), C.POINTER(CCamera), C.POINTER(CParams),
                                 C.POINTER(CViewState), vp]
    lib.fhgs_bin_sort.argtypes = [vp, C.POINTER(CCamera), C.POINTER(CViewState), C.POINTER(C.c_uint64),
                                  C.c_uint32, vp]
    lib.fhgs_render.argtypes = [vp, C.POINTER(CGaussians), C.POINTER(CCamera), C.POINTER(CParams),
                                C.POINTER(CViewState), vp, vp, vp, vp, vp]
    lib.fhgs_fuse_features.argtypes = [vp, C.POINTER(CCamera), C.POINTER(CParams), C.POINTER(CViewState), vp,
                                       C.c_int32, C.c_int32, vp, vp, vp, C.c_int32, C.c_uint32, vp]
    lib.fhgs_frame_host.argtypes = [vp, C.POINTER(CHostFrame), C.POINTER(CGaussians), C.POINTER(CCamera),
                                    C.POINTER(CParams), C.POINTER(CViewState), C.POINTER(CFrameWorkspace),
                                    C.POINTER(C.c_uint64), vp]
    lib.fhgs_ndfd_forward.argtypes = [vp, C.POINTER(CGaussians), C.POINTER(CCamera), C.POINTER(CParams), C.POINTER(CViewState),
                                      vp, C.c_int32, C.c_float, C.c_float, C.c_int32, vp, vp, vp]
    lib.fhgs_ndfd_backward_work_bytes.restype = C.c_size_t
    lib.fhgs_ndfd_backward_work_bytes.argtypes = [C.c_int32, C.c_int32, C.c_int32]
    lib.fhgs_ndfd_backward.argtypes = [vp, C.POINTER(CGaussians), C.POINTER(CCamera), C.POINTER(CParams), C.POINTER(CViewState),
                                       vp, C.c_int32, C.c_float, C.c_float, C.c_float, C.c_float, vp, vp, C.c_size_t, vp]
    lib.fhgs_ffma_peak.argtypes = [vp, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_double), vp]
    lib.fhgs_scan_offsets_static_max_n.restype = C.c_int32
    lib.fhgs_scan_offsets_static_max_n.argtypes = []
    lib.fhgs_scan_offsets_static.argtypes = [vp, vp, C.c_int32, vp, vp, vp]
    lib.fhgs_render_fuse.argtypes = [vp, C.POINTER(CGaussians), C.POINTER(CCamera), C.POINTER(CParams), C.POINTER(CViewState),
                                     vp, vp, vp, vp, vp, vp, vp, vp]
    return lib


lib = _load()


def version() -> str:
    return lib.fhgs_version().decode()


def default_params(**overrides) -> CParams:
    p = CParams()
    lib.fhgs_default_params(C.byref(p))
    for k, v in overrides.items():
        if k == "bg":
            p.bg[0], p.bg[1], p.bg[2] = [float(x) for x in v]
        elif k in ("rect_mode", "primitive"):
            setattr(p, k, int(v))
        else:
            setattr(p, k, float(v))
    return p


def make_camera(view, proj, cam_pos, width: int, height: int) -> CCamera:
    c = CCamera()
    v = np.asarray(view, np.float32).ravel()
    pj = np.asarray(proj, np.float32).ravel()
    cp = np.asarray(cam_pos, np.float32).ravel()
    for i in range(16):
        c.view[i] = float(v[i])
        c.proj[i] = float(pj[i])
    for i in range(3):
        c.cam_pos[i] = float(cp[i])
    c.width, c.height = int(width), int(height)
    return c


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def _dtype_code(t: torch.Tensor) -> int:
    if t.dtype == torch.float32:
        return FHGS_F32
    if t.dtype == torch.float16:
        return FHGS_F16
    if t.dtype == torch.bfloat16:
        return FHGS_BF16   # fhgs_render / fhgs_fuse_features / fhgs_frame_host only
    raise TypeError(f"unsupported feature dtype {t.dtype}")


class Context:
    def __init__(self, device: int = 0):
        if not torch.cuda.is_available():
            raise RuntimeError("fhgs needs a CUDA device (sm_100a); there is no CPU fallback")
        self.device = int(device)
        torch.cuda.set_device(self.device)
        torch.cuda.init()
        h = C.c_void_p()
        st = lib.fhgs_create(C.byref(h), self.device)
        if st != FHGS_OK:
            raise FhgsError(st, "fhgs_create failed (no suitable device?)")
        self.handle = h

    def close(self):
        if getattr(self, "handle", None):
            lib.fhgs_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_diagnostics(self, enable: bool):
        """fhgs_set_diagnostics: make fhgs_render fill ViewState.tile_visited() (work accounting only)."""
        lib.fhgs_set_diagnostics(self.handle, 1 if enable else 0)

    def check(self, st: int):
        if st != FHGS_OK:
            raise FhgsError(st, lib.fhgs_last_error(self.handle).decode())

    def ffma_peak(self, iters: int = 4096):
        ops, ms = C.c_double(), C.c_double()
        self.check(lib.fhgs_ffma_peak(self.handle, iters, C.byref(ops), C.byref(ms), _stream(None)))
        return ops.value, ms.value


class Gaussians:
    """Device copy of a scene (torch tensors) plus the C struct that points at them."""

    def __init__(self, mean, scale, quat, opacity, sh, feat, sh_degree: int, device="cuda"):
        def dev(a, dt):
            if a is None:
                return None
            t = a if isinstance(a, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(a))
            return t.to(device=device, dtype=dt).contiguous()
        self.mean, self.scale, self.quat = dev(mean, torch.float32), dev(scale, torch.float32), dev(quat, torch.float32)
        self.opacity, self.sh = dev(opacity, torch.float32), dev(sh, torch.float32)
        if feat is None:
            self.feat = None
        else:
            fdt = feat.dtype if isinstance(feat, torch.Tensor) else torch.from_numpy(np.asarray(feat)[:0]).dtype
            self.feat = dev(feat, fdt)
        self.sh_degree = int(sh_degree)
        self.n = int(self.mean.shape[0])
        self.c = CGaussians()
        self.refresh()

    def refresh(self):
        c = self.c
        c.n, c.sh_degree = self.n, self.sh_degree
        c.feat_dim = 0 if self.feat is None else int(self.feat.shape[1])
        c.feat_dtype = FHGS_F32 if self.feat is None else _dtype_code(self.feat)
        c.mean, c.scale, c.quat = self.mean.data_ptr(), self.scale.data_ptr(), self.quat.data_ptr()
        c.opacity, c.sh = self.opacity.data_ptr(), self.sh.data_ptr()
        c.feat = None if self.feat is None else self.feat.data_ptr()


class ViewState:
    """Caller-owned per-view buffers (fhgs_view_state)."""

    def __init__(self, n: int, width: int, height: int, capacity: int, device="cuda", surfel: bool = False):
        self.n, self.width, self.height, self.capacity = int(n), int(width), int(height), int(capacity)
        gw, gh = (width + 15) // 16, (height + 15) // 16
        z = lambda shape, dt: torch.zeros(shape, dtype=dt, device=device)
        m = max(self.n, 1)
        self.xy, self.depth = z((m, 2), torch.float32), z((m,), torch.float32)
        self.conic_opacity, self.rgb = z((m, 4), torch.float32), z((m, 3), torch.float32)
        self.radius = z((m,), torch.int32)
        self.rect = z((m, 4), torch.int16)            # uint16 payload
        self.tiles_touched = z((m,), torch.int32)      # uint32 payload
        self.offsets = z((m,), torch.int32)            # uint32 payload
        self.num_instances = z((1,), torch.int64)
        cap = max(self.capacity, 1)
        self.keys = [z((cap,), torch.int64), z((cap,), torch.int64)]
        self.vals = [z((cap,), torch.int32), z((cap,), torch.int32)]
        self.ranges = z((gw * gh, 2), torch.int32)
        sb = int(lib.fhgs_scratch_bytes(self.n, self.width, self.height, self.capacity))
        self.scratch = z((sb + 256,), torch.uint8)
        c = self.c = CViewState()
        c.n, c.width, c.height, c.sorted_buf, c.capacity = self.n, self.width, self.height, 0, self.capacity
        c.xy, c.depth, c.conic_opacity, c.rgb = (self.xy.data_ptr(), self.depth.data_ptr(),
                                                 self.conic_opacity.data_ptr(), self.rgb.data_ptr())
        c.radius, c.rect, c.tiles_touched = self.radius.data_ptr(), self.rect.data_ptr(), self.tiles_touched.data_ptr()
        c.offsets, c.num_instances = self.offsets.data_ptr(), self.num_instances.data_ptr()
        c.keys[0], c.keys[1] = self.keys[0].data_ptr(), self.keys[1].data_ptr()
        c.vals[0], c.vals[1] = self.vals[0].data_ptr(), self.vals[1].data_ptr()
        c.ranges = self.ranges.data_ptr()
        sp = self.scratch.data_ptr()
        c.scratch = (sp + 255) // 256 * 256
        c.scratch_bytes = sb
        self.ray_transform = z((m, 12), torch.float32) if surfel else None     # FHGS_PRIM_SURFEL only
        c.ray_transform = self.ray_transform.data_ptr() if surfel else None

    def tile_visited(self) -> torch.Tensor:
        """Diagnostics written by fhgs_render (see fhgs_scratch_tile_visited): int32 tensor [GW*GH] (device)."""
        off = int(lib.fhgs_scratch_tile_visited(self.n, self.width, self.height, self.capacity))
        base = self.c.scratch - self.scratch.data_ptr()
        gw, gh = (self.width + 15) // 16, (self.height + 15) // 16
        return self.scratch[base + off: base + off + 4 * gw * gh].view(torch.int32)

    # views of the results with the library's integer types (numpy, host)
    def sorted_keys(self, m: int) -> np.ndarray:
        return self.keys[self.c.sorted_buf][:m].cpu().numpy().view(np.uint64)

    def sorted_vals(self, m: int) -> np.ndarray:
        return self.vals[self.c.sorted_buf][:m].cpu().numpy().view(np.uint32)

    def projected(self) -> dict:
        n = self.n
        return dict(xy=self.xy[:n].cpu().numpy(), depth=self.depth[:n].cpu().numpy(),
                    conic_opacity=self.conic_opacity[:n].cpu().numpy(), rgb=self.rgb[:n].cpu().numpy(),
                    radius=self.radius[:n].cpu().numpy(), rect=self.rect[:n].cpu().numpy().view(np.uint16),
                    tiles_touched=self.tiles_touched[:n].cpu().numpy().view(np.uint32),
                    **({} if self.ray_transform is None else {"ray_transform": self.ray_transform[:n].cpu().numpy()}))


def project(ctx: Context, g: Gaussians, cam: CCamera, prm: CParams, vs: ViewState, stream=None):
    """fhgs_project (step P)."""
    ctx.check(lib.fhgs_project(ctx.handle, C.byref(g.c), C.byref(cam), C.byref(prm), C.byref(vs.c), _stream(stream)))


def bin_sort(ctx: Context, cam: CCamera, vs: ViewState, sync: bool = False, flags: int = 0, stream=None):
    """fhgs_bin_sort (step S).  sync=True returns M (and raises FhgsError(CAPACITY) on overflow)."""
    m = C.c_uint64(0)
    st = lib.fhgs_bin_sort(ctx.handle, C.byref(cam), C.byref(vs.c), C.byref(m) if sync else None,
                           C.c_uint32(flags), _stream(stream))
    ctx.check(st)
    return int(m.value) if sync else None


def scan_offsets_static(ctx: Context, tiles_touched, offsets, num_instances=None, n=None, stream=None):
    """fhgs_scan_offsets_static: the allocation-free prefix sum of step S1 (library-owned static scratch).
    tiles_touched / offsets: uint32-sized device tensors [n]; num_instances: optional 8-byte device tensor [1]."""
    n = int(tiles_touched.numel()) if n is None else int(n)
    ctx.check(lib.fhgs_scan_offsets_static(ctx.handle, _ptr(tiles_touched), n, _ptr(offsets), _ptr(num_instances),
                                           _stream(stream)))


def render(ctx: Context, g: Gaussians, cam: CCamera, prm: CParams, vs: ViewState, out_rgb, out_feat=None,
           out_T=None, out_ncontrib=None, stream=None):
    """fhgs_render (step R).  Outputs are caller-allocated torch tensors."""
    ctx.check(lib.fhgs_render(ctx.handle, C.byref(g.c), C.byref(cam), C.byref(prm), C.byref(vs.c), _ptr(out_rgb),
                              _ptr(out_feat), _ptr(out_T), _ptr(out_ncontrib), _stream(stream)))


def render_fuse(ctx: Context, g: Gaussians, cam: CCamera, prm: CParams, vs: ViewState, out_rgb, out_feat, gt, num, den,
                out_T=None, out_ncontrib=None, stream=None):
    """fhgs_render_fuse: steps R and F in one traversal (per-pixel regime: D not a multiple of 64).  gt has the dtype of
    the feature rows; num / den are accumulated into, not cleared."""
    if gt.dtype != g.feat.dtype:
        raise TypeError("gt must have the storage type of the feature rows")
    ctx.check(lib.fhgs_render_fuse(ctx.handle, C.byref(g.c), C.byref(cam), C.byref(prm), C.byref(vs.c), _ptr(out_rgb),
                                   _ptr(out_feat), _ptr(out_T), _ptr(out_ncontrib), _ptr(gt), _ptr(num), _ptr(den),
                                   _stream(stream)))


def fuse_features(ctx: Context, cam, prm: CParams, vs: ViewState, gt, num, den, out_feat=None, flags: int = 0,
                  stream=None):
    """fhgs_fuse_features (step F).  gt [H,W,D] f32/f16/bf16; num [n,D] f32; den [n] f32."""
    d = int(num.shape[1])
    gt_code = FHGS_F32 if gt is None else _dtype_code(gt)
    out_code = FHGS_F32 if out_feat is None else _dtype_code(out_feat)
    ctx.check(lib.fhgs_fuse_features(ctx.handle, None if cam is None else C.byref(cam), C.byref(prm), C.byref(vs.c),
                                     _ptr(gt), d, gt_code, _ptr(num), _ptr(den), _ptr(out_feat), out_code,
                                     C.c_uint32(flags), _stream(stream)))


def ndfd_forward(ctx: Context, g: Gaussians, cam: CCamera, prm: CParams, vs: ViewState, gt, out_lgt, out_lcf,
                 k: float = 20.0, lam: float = 0.5, mode: int = 0, stream=None):
    """fhgs_ndfd_forward: per-pixel L_gt, L_cf ([H,W] f32 tensors, caller-allocated) of PAPER.md Eq. 5-6.
    mode: FHGS_NDFD_BLEND_ORDER (0) or FHGS_NDFD_FAR_TO_NEAR (1)."""
    ctx.check(lib.fhgs_ndfd_forward(ctx.handle, C.byref(g.c), C.byref(cam), C.byref(prm), C.byref(vs.c), _ptr(gt),
                                    _dtype_code(gt), C.c_float(k), C.c_float(lam), C.c_int32(mode), _ptr(out_lgt),
                                    _ptr(out_lcf), _stream(stream)))


def ndfd_backward(ctx: Context, g: Gaussians, cam: CCamera, prm: CParams, vs: ViewState, gt, grad_opacity,
                  k: float = 20.0, lam: float = 0.5, lam1: float = 1.0, lam2: float = 1.0, work=None, stream=None):
    """fhgs_ndfd_backward: accumulates dL/d opacity into grad_opacity [n] f32.  `work`: optional uint8 scratch tensor
    (allocated here when None); returned for reuse."""
    nbytes = int(lib.fhgs_ndfd_backward_work_bytes(vs.width, vs.height, g.c.feat_dim))
    if work is None or work.numel() < nbytes + 256:
        work = torch.empty((nbytes + 256,), dtype=torch.uint8, device=grad_opacity.device)
    wp = (work.data_ptr() + 255) // 256 * 256
    ctx.check(lib.fhgs_ndfd_backward(ctx.handle, C.byref(g.c), C.byref(cam), C.byref(prm), C.byref(vs.c), _ptr(gt),
                                     _dtype_code(gt), C.c_float(k), C.c_float(lam), C.c_float(lam1), C.c_float(lam2),
                                     _ptr(grad_opacity), C.c_void_p(wp), C.c_size_t(nbytes), _stream(stream)))
    return work


def frame_host(ctx: Context, host: dict, g: Gaussians, cam: CCamera, prm: CParams, vs: ViewState, ws: dict,
               stream=None) -> int:
    """fhgs_frame_host: one whole frame from HOST (pinned) tensors; returns M."""
    hf = CHostFrame()
    for k in ("mean", "scale", "quat", "opacity", "sh", "feat", "gt", "out_rgb", "out_feat", "fused_feat"):
        t = host.get(k)
        setattr(hf, k, None if t is None else t.data_ptr())
    w = CFrameWorkspace()
    for k in ("out_rgb", "out_feat", "gt", "num", "den", "fused_feat"):
        setattr(w, k, ws[k].data_ptr())
    m = C.c_uint64(0)
    ctx.check(lib.fhgs_frame_host(ctx.handle, C.byref(hf), C.byref(g.c), C.byref(cam), C.byref(prm), C.byref(vs.c),
                                  C.byref(w), C.byref(m), _stream(stream)))
    return int(m.value)

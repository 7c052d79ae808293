"""The whole frame (P -> S -> R -> F, including fhgs_bin_sort's fork / join onto the context's side stream) can be
captured into a CUDA graph: no entry point synchronises, allocates or touches the legacy stream on the way.  The replayed
graph must reproduce the stream-ordered calls: integers and the rendered images bit for bit, the fused accumulators up to
the order of their floating-point atomics."""
import numpy as np
import pytest

from paper_2505_19154_b200 import inputs
import parity_util as pu

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("case", ["tiny", "d128"])
def test_frame_captured_in_cuda_graph(case):
    import torch
    from paper_2505_19154_b200 import binding as fb
    cfg = inputs.CONFIGS["tiny"] if case == "tiny" else inputs.scaled(inputs.CONFIGS["mid"], n=30_000, width=200, height=120,
                                                                      log_scale_mu=-3.0)
    scene = inputs.make_scene(cfg)
    cam_h = inputs.make_camera(cfg, 0)
    W, H, D, n = cfg.width, cfg.height, cfg.feat_dim, scene.n
    ctx = fb.Context(0)
    g = fb.Gaussians(scene.mean, scene.scale, scene.quat, scene.opacity, scene.sh, scene.feat, scene.sh_degree)
    cam = fb.make_camera(cam_h.view, cam_h.proj, cam_h.cam_pos, cam_h.width, cam_h.height)
    prm = fb.default_params()
    vs0 = fb.ViewState(n, W, H, 0)
    fb.project(ctx, g, cam, prm, vs0)
    torch.cuda.synchronize()
    M = int(vs0.tiles_touched.to(torch.int64).sum())
    vs = fb.ViewState(n, W, H, M + 1024)
    dev = g.mean.device
    gt = torch.from_numpy(inputs.make_gt_map(cfg, 0, cam_h)).to(dev)
    out = dict(rgb=torch.empty((H, W, 3), device=dev), feat=torch.empty((H, W, D), device=dev),
               T=torch.empty((H, W), device=dev), n=torch.empty((H, W), dtype=torch.int32, device=dev),
               num=torch.zeros((n, D), device=dev), den=torch.zeros((n,), device=dev), fused=g.feat.clone())

    def frame(stream):
        fb.project(ctx, g, cam, prm, vs, stream=stream)
        fb.bin_sort(ctx, cam, vs, stream=stream)   # no host read-back of M: nothing synchronises
        fb.render(ctx, g, cam, prm, vs, out["rgb"], out["feat"], out["T"], out["n"], stream=stream)
        fb.fuse_features(ctx, cam, prm, vs, gt, out["num"], out["den"], out["fused"],
                         fb.FHGS_FUSE_ZERO | fb.FHGS_FUSE_FINALIZE, stream=stream)

    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        frame(s)
        s.synchronize()
        ref = {k: v.clone() for k, v in out.items()}
        ref_int = dict(offsets=vs.offsets.clone(), ranges=vs.ranges.clone(), m=vs.num_instances.clone(),
                       vals=vs.vals[vs.c.sorted_buf][:M].clone(), keys=vs.keys[vs.c.sorted_buf][:M].clone())
        assert int(ref_int["m"].item()) == M > 0
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=s):
            frame(torch.cuda.current_stream())
        for rep in range(2):
            for k in ("rgb", "feat", "T", "num", "den"):
                out[k].fill_(float("nan"))
            out["n"].fill_(-1)
            out["fused"].copy_(g.feat)
            vs.vals[vs.c.sorted_buf].fill_(-1)
            graph.replay()
            s.synchronize()
            for k in ("rgb", "feat", "T", "n"):
                assert torch.equal(out[k], ref[k]), f"{k} differs after replay {rep}"
            assert torch.equal(vs.offsets, ref_int["offsets"]) and torch.equal(vs.ranges, ref_int["ranges"])
            assert torch.equal(vs.vals[vs.c.sorted_buf][:M], ref_int["vals"])
            assert torch.equal(vs.keys[vs.c.sorted_buf][:M], ref_int["keys"])
            gmax = float(gt.abs().max())
            dden = (out["den"] - ref["den"]).abs()
            assert bool((dden <= pu.TOL_F32 * ref["den"].abs() + 1e-12).all())
            dnum = (out["num"] - ref["num"]).abs().amax(dim=1)
            assert bool((dnum <= pu.TOL_F32 * ref["den"].abs() * gmax + 1e-12).all())
            assert float((out["fused"] - ref["fused"]).abs().max()) <= pu.TOL_F32

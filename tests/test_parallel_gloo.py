"""N > 1 host logic on CPU: world_size-2 `gloo` process groups exercise paper_2505_19154_b200.parallel
(view sharding, the one all-reduce of the fusion accumulators, max-over-ranks timing).  Each rank fuses its
share of the Tiny config's views with the CPU oracle (tests may use oracle/); the all-reduced accumulators
must equal a single-process fusion of all views."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import fhgs_oracle as fo
from paper_2505_19154_b200 import inputs, parallel
import parity_util as pu


def _free_port() -> int:
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _oracle_view_fuser(cfg, scene):
    def fuse(v, num, den):
        cam = inputs.make_camera(cfg, v)
        pr = pu.oracle_view(scene, cam)
        order = fo.global_order(pr)
        gt = inputs.make_gt_map(cfg, v, cam)
        fo.fuse(pr, order, gt, cfg.width, cfg.height, num=num, den=den)
    return fuse


def _worker(rank, world, port, n_views, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = inputs.CONFIGS["tiny"]
        scene = inputs.make_scene(cfg)
        fuse = _oracle_view_fuser(cfg, scene)
        num = torch.full((scene.n, cfg.feat_dim), 7.0, dtype=torch.float64)   # garbage: ZERO must clear it
        den = torch.full((scene.n,), 7.0, dtype=torch.float64)
        state = {}

        def fuse_one_view(v, first):
            if first:
                num.zero_()
                den.zero_()
            fuse(v, num.numpy(), den.numpy())   # numpy views share the tensors' memory

        def finalize():
            state["feat"] = fo.finalize(num.numpy(), den.numpy(), scene.feat.astype(np.float32))

        def before_reduce():    # bench.py records its CUDA event here: must run once, after the last view, before finalize
            assert "feat" not in state
            state["hook"] = state.get("hook", 0) + 1

        mine = parallel.fuse_views_sharded(list(range(n_views)), fuse_one_view, num, den, finalize, before_reduce=before_reduce)
        assert state["hook"] == 1
        t = parallel.max_over_ranks(10.0 + rank)
        np.savez(os.path.join(out_dir, f"rank{rank}.npz"), num=num.numpy(), den=den.numpy(), feat=state["feat"],
                 mine=np.array(mine, dtype=np.int64), t=np.array([t]))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_views", [4, 1])
def test_view_sharded_fusion_world2(tmp_path, n_views):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), n_views, str(tmp_path)), nprocs=world, join=True)
    cfg = inputs.CONFIGS["tiny"]
    scene = inputs.make_scene(cfg)
    fuse = _oracle_view_fuser(cfg, scene)
    num = np.zeros((scene.n, cfg.feat_dim))
    den = np.zeros(scene.n)
    for v in range(n_views):
        fuse(v, num, den)
    feat = fo.finalize(num, den, scene.feat.astype(np.float32))
    seen = []
    for r in range(world):
        z = np.load(os.path.join(str(tmp_path), f"rank{r}.npz"))
        seen += z["mine"].tolist()
        # every rank ends with the accumulators of ALL views (sum order differs: fp64 round-off only)
        np.testing.assert_allclose(z["num"], num, rtol=1e-12, atol=1e-13)
        np.testing.assert_allclose(z["den"], den, rtol=1e-12, atol=1e-13)
        np.testing.assert_allclose(z["feat"], feat, rtol=1e-9, atol=1e-12)
        assert float(z["t"][0]) == 11.0   # max over ranks of 10 + rank
    assert sorted(seen) == list(range(n_views))   # every view fused exactly once


def test_shard_views_partition():
    for n, world in [(200, 8), (200, 3), (5, 8), (0, 2), (7, 1)]:
        parts = [parallel.shard_views(n, r, world) for r in range(world)]
        flat = sorted(v for p in parts for v in p)
        assert flat == list(range(n))
        assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
    with pytest.raises(ValueError):
        parallel.shard_views(4, 2, 2)


def test_single_process_is_identity():
    num = torch.ones(3, 4, dtype=torch.float64)
    den = torch.ones(3, dtype=torch.float64)
    parallel.allreduce_accumulators(num, den)
    assert parallel.max_over_ranks(3.5) == 3.5 and parallel.world_info() == (0, 1)
    assert float(num.sum()) == 12.0

"""fhgs_scan_offsets_static (the allocation-free prefix sum of step S1, library-owned static scratch) against the
existing path (fhgs_bin_sort's offsets / num_instances, caller scratch): integer work, bit-exact.  Collected last
on purpose (pytest -x): a failure here must not hide another test."""
import numpy as np
import pytest

from paper_2505_19154_b200 import inputs


def _scene_case(n, width, height):
    import parity_util as pu
    cfg = inputs.scaled(inputs.CONFIGS["small"], n=n, width=width, height=height)
    scene = inputs.make_scene(cfg)
    cam = inputs.make_camera(cfg, 0)
    gp = pu.GpuPath(scene, width, height, 64 * n + 4096)
    gp.project_sort(cam)          # existing path: fills vs.tiles_touched, vs.offsets, vs.num_instances
    return gp


@pytest.mark.gpu
def test_static_scratch_scan_matches_bin_sort_two_calls_in_a_row():
    import torch
    from paper_2505_19154_b200 import binding as fb
    # 37 look-back tiles with a ragged tail, then a shorter input: the second call must not see the first call's status words
    gp_a = _scene_case(37 * 1024 + 391, 256, 256)
    gp_b = _scene_case(5 * 1024 + 7, 128, 96)
    for rep in range(2):
        for gp in (gp_a, gp_b):
            vs = gp.vs
            off = torch.full_like(vs.offsets, -1)
            m = torch.full_like(vs.num_instances, -1)
            fb.scan_offsets_static(gp.ctx, vs.tiles_touched, off, m, n=vs.n)
            torch.cuda.synchronize()
            assert torch.equal(off[:vs.n], vs.offsets[:vs.n]), f"offsets differ (rep {rep}, n {vs.n})"
            assert int(m.item()) == int(vs.num_instances.item()) > 0
            # and against the plain definition (uint32 wrap-around like the library's)
            ref = np.cumsum(vs.tiles_touched[:vs.n].cpu().numpy().view(np.uint32).astype(np.uint64))
            assert np.array_equal(off[:vs.n].cpu().numpy().view(np.uint32), ref.astype(np.uint32))
            assert int(m.item()) == int(ref[-1])


@pytest.mark.gpu
def test_static_scratch_scan_limits_and_empty():
    import torch
    from paper_2505_19154_b200 import binding as fb
    ctx = fb.Context(0)
    max_n = int(fb.lib.fhgs_scan_offsets_static_max_n())
    assert max_n == 1 << 22
    # the largest size the static array serves, every look-back word in use
    tt = torch.randint(0, 50, (max_n,), dtype=torch.int32, device="cuda")
    off = torch.empty_like(tt)
    m = torch.zeros((1,), dtype=torch.int64, device="cuda")
    for _ in range(2):
        off.fill_(-1)
        fb.scan_offsets_static(ctx, tt, off, m)
        torch.cuda.synchronize()
        ref = torch.cumsum(tt.to(torch.int64), 0)
        assert torch.equal(off.to(torch.int64), ref) and int(m.item()) == int(ref[-1].item())
    # beyond the maximum: a clear error, nothing enqueued
    big = torch.zeros((max_n + 1,), dtype=torch.int32, device="cuda")
    with pytest.raises(fb.FhgsError) as e:
        fb.scan_offsets_static(ctx, big, big.clone(), m)
    assert e.value.status == fb.FHGS_ERR_INVALID and "static scratch" in str(e.value)
    # empty input: only M = 0 is written
    m.fill_(-1)
    fb.scan_offsets_static(ctx, None, None, m, n=0)
    torch.cuda.synchronize()
    assert int(m.item()) == 0

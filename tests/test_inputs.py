"""Host-side checks of the seeded input generators (no method arithmetic lives there)."""
import numpy as np

from paper_2505_19154_b200 import inputs


def test_round_to_bf16_matches_torch_and_ties_to_even():
    import torch
    rng = np.random.default_rng(5)
    a = np.concatenate([rng.standard_normal(100_000).astype(np.float32) * np.float32(10.0) ** rng.integers(-6, 6, 100_000),
                        np.array([0.0, -0.0, 1.0, -1.0, 3.0e38, 1e-40, -1e-40], dtype=np.float32)])
    # exact ties: 1 + (2k+1) * 2^-9 lies half-way between two bf16 values
    ties = (1.0 + (2 * np.arange(64) + 1) * 2.0 ** -9).astype(np.float32)
    a = np.concatenate([a, ties, -ties])
    r = inputs.round_to_bf16(a)
    t = torch.from_numpy(a).to(torch.bfloat16).to(torch.float32).numpy()
    assert np.array_equal(r.view(np.uint32), t.view(np.uint32))
    assert np.all((r.view(np.uint32) & 0xFFFF) == 0)                       # representable in bfloat16
    assert np.array_equal(inputs.round_to_bf16(r).view(np.uint32), r.view(np.uint32))   # idempotent


def test_bf16_configs_carry_representable_values():
    cfg = inputs.scaled(inputs.CONFIGS["tiny"], feat_dtype="bf16")
    scene = inputs.make_scene(cfg)
    gt = inputs.make_gt_map(cfg, 0, inputs.make_camera(cfg, 0))
    for arr in (scene.feat, gt):
        assert arr.dtype == np.float32 and np.all((arr.view(np.uint32) & 0xFFFF) == 0)
    # same seed, same draws: the bf16 scene is the rounded f32 scene
    ref = inputs.make_scene(inputs.CONFIGS["tiny"])
    assert np.array_equal(scene.feat, inputs.round_to_bf16(ref.feat))

"""GPU-vs-oracle parity of ggt_guidance_features (A.4 items 5-8) through the C ABI (-m gpu):
bit-identical feature tensors on the configs' shapes, on depth maps with holes and ragged sizes."""
import numpy as np
import pytest

import oracle
from paper_2505_18932_b200 import synth

pytestmark = pytest.mark.gpu


def run(tgt, depth, views):
    import torch
    from paper_2505_18932_b200 import binding
    of = oracle.features(tgt, depth, views)
    ctx = binding.Context()
    out = torch.full((4 * len(views), tgt.height, tgt.width), -7.0, dtype=torch.float32, device="cuda")
    ctx.ggt_guidance_features(tgt, torch.from_numpy(np.ascontiguousarray(depth)).cuda(), views, out)
    torch.cuda.synchronize()
    g = out.cpu().numpy()
    bad = g.view(np.uint32) != of.view(np.uint32)
    assert not bad.any(), "%d of %d feature values differ (channels %s)" % (bad.sum(), bad.size, np.unique(np.nonzero(bad)[0])[:8])
    return of


def guidance_depth(wl, tgt, rng, holes=0.03):
    d = synth.noisy_depth(synth.raycast(tgt, wl.scene)[0], 77, 0, 0.005, 0.0).astype(np.float32)
    d[rng.uniform(size=d.shape) < holes] = 0
    return d


@pytest.mark.parametrize("name,scale", [("C1", 1.0), ("C2", 1.0), ("C3", 1.0), ("C4", 0.5), ("C5", 0.5)])
def test_features_configs(name, scale):
    wl = synth.workload(name, scale=scale)
    tgt = wl.targets(0)[0]
    views = [wl.rig[v] for v in wl.views_for(tgt)]
    of = run(tgt, guidance_depth(wl, tgt, np.random.default_rng(3)), views)
    K = len(views)
    assert (of[:K] != 0).mean() > 0.8 and np.all(np.abs(of[:2 * K]) <= 1 + 1e-6)


@pytest.mark.parametrize("n_views,W,H", [(1, 33, 9), (3, 70, 37), (16, 64, 48)])
def test_features_ragged_and_holes(n_views, W, H):
    wl = synth.workload("C2", scale=0.2)
    rig = synth.grid_rig(W + 13, H + 6)
    tgt = synth.camera_from_pose((0.04, -0.03, 0.01), synth.rot_yaw_pitch(0.02, 0.01), 0.8 * W, 0.8 * W, W / 2, H / 2, W, H)
    views = [rig[i] for i in synth.nearest_views(tgt, rig, n_views)]
    rng = np.random.default_rng(W)
    run(tgt, guidance_depth(wl, tgt, rng, holes=0.3), views)          # many one-sided differences and undefined pixels
    run(tgt, np.zeros((H, W), np.float32), views)                     # no depth at all
    d = np.zeros((H, W), np.float32); d[H // 2, W // 2] = 2.0
    assert np.all(run(tgt, d, views)[:2 * n_views] == 0)


def test_features_error_codes():
    import torch
    from paper_2505_18932_b200 import binding
    ctx = binding.Context()
    cam = synth.camera_from_pose((0, 0, 0), np.eye(3), 30, 30, 16.5, 4.5, 33, 9)
    d = torch.full((9, 33), 2.0, device="cuda")
    out = torch.empty((4, 9, 33), device="cuda")
    ctx.ggt_guidance_features(cam, d, [cam], out)
    torch.cuda.synchronize()
    assert torch.all((out[1] - 1.0).abs() < 1e-6) and torch.all(out[2] == 0.0) and torch.all(out[3] == 1.0) and torch.all(out[0] < 0)
    with pytest.raises(binding.GgtError):
        ctx.ggt_guidance_features(cam, d, [], out)
    with pytest.raises(binding.GgtError):
        ctx.ggt_guidance_features(cam, d, [cam] * 17, out)

"""GPU-vs-oracle parity of ggt_splat_forward / ggt_temporal_weight_mask through the C ABI.

Both sides evaluate readings S1-S8 in the same fp32 operation order (including the exponential, S8), so every output is
compared bit for bit: opacity, premultiplied colour, normalised depth, splatted mask and the per-pixel list length.
"""
import numpy as np
import pytest

import oracle
from paper_2505_18932_b200 import synth

pytestmark = pytest.mark.gpu


def gpu_splat(ctx, tgt, src, depth, rgb=None, mask=None, **kw):
    import torch
    Ht, Wt = tgt.height, tgt.width
    g = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()
    out = dict(rgb=torch.empty((3, Ht, Wt), device="cuda") if rgb is not None else None,
               alpha=torch.empty((Ht, Wt), device="cuda"), depth=torch.empty((Ht, Wt), device="cuda"),
               mask=torch.empty((Ht, Wt), device="cuda") if mask is not None else None,
               count=torch.empty((Ht, Wt), dtype=torch.int32, device="cuda"))
    ctx.ggt_splat_forward(tgt, src, g(depth), rgb=g(rgb), mask=g(mask), out_rgb=out["rgb"], out_alpha=out["alpha"],
                          out_depth=out["depth"], out_mask=out["mask"], out_count=out["count"], **kw)
    torch.cuda.synchronize()
    return {k: (None if v is None else v.cpu().numpy()) for k, v in out.items()}


def assert_same(o, g):
    assert np.array_equal(o["count"], g["count"])
    for k in ("alpha", "depth", "rgb", "mask"):
        if o[k] is None:
            continue
        assert np.array_equal(o[k].view(np.uint32), g[k].view(np.uint32)), (k, float(np.abs(o[k] - g[k]).max()))


def cam(centre=(0, 0, 0), R=None, f=100.0, W=40, H=30):
    return synth.camera_from_pose(centre, np.eye(3) if R is None else R, f, f, W / 2, H / 2, W, H)


@pytest.mark.parametrize("case", ["rotated", "ties", "single", "empty"])
def test_splat_small_cases_bit_exact(case):
    from paper_2505_18932_b200 import binding
    rng = np.random.default_rng(11)
    W, H = 37, 29                                                  # ragged sizes: several CTAs and a tail in both images
    src = cam(centre=(0.05, -0.02, 0.0), R=synth.rot_yaw_pitch(0.03, -0.02), f=40.0, W=W, H=H)
    tgt = cam(centre=(-0.12, 0.06, 0.25), R=synth.rot_yaw_pitch(-0.08, 0.05), f=52.0, W=45, H=35)
    depth = rng.uniform(1.0, 3.0, (H, W)).astype(np.float32)
    depth[rng.uniform(size=(H, W)) < 0.1] = 0
    if case == "ties":
        src, tgt = cam(f=40.0, W=W, H=H), cam(centre=(0.07, 0.0, 0.0), f=40.0, W=45, H=35)
        depth = np.where(rng.uniform(size=(H, W)) < 0.5, 1.5, 2.25).astype(np.float32)
    elif case == "single":
        depth[:] = 0; depth[14, 20] = 2.0
    elif case == "empty":
        depth[:] = 0
    rgb = rng.integers(0, 256, (H, W, 3), dtype=np.uint8)
    mask = rng.uniform(0.6, 1.0, (H, W)).astype(np.float32)
    ctx = binding.Context()
    o = oracle.splat_forward(tgt, src, depth, rgb=rgb, mask=mask)
    g = gpu_splat(ctx, tgt, src, depth, rgb=rgb, mask=mask)
    assert_same(o, g)
    last, need = ctx.ggt_splat_status()
    assert last == int(o["count"].sum()) and need == 0
    if case == "rotated":
        assert (o["alpha"] > 0.5).mean() > 0.3
        # 4-byte colour pixels, other parameters, outputs left out
        rgba = np.concatenate([rgb, np.zeros((H, W, 1), np.uint8)], axis=2)
        o2 = oracle.splat_forward(tgt, src, depth, rgb=rgba, sigma_px=0.7, dilation=0.1, z_cull=1.2)
        g2 = gpu_splat(ctx, tgt, src, depth, rgb=rgba, sigma_px=0.7, dilation=0.1, z_cull=1.2)
        assert_same(o2, g2)
        assert not np.array_equal(o2["alpha"], o["alpha"])


def test_splat_capacity_overflow_is_reported_and_recoverable():
    from paper_2505_18932_b200 import binding
    rng = np.random.default_rng(2)
    src, tgt = cam(f=40.0, W=48, H=32), cam(centre=(0.05, 0, 0), f=40.0, W=48, H=32)
    depth = rng.uniform(1.5, 2.0, (32, 48)).astype(np.float32)
    ctx = binding.Context()
    o = oracle.splat_forward(tgt, src, depth)
    total = int(o["count"].sum())
    ctx.ggt_splat_reserve(total // 2)
    g = gpu_splat(ctx, tgt, src, depth)
    last, need = ctx.ggt_splat_status()
    assert last == total and need == total                         # the call says how many entries it needed
    assert float(np.abs(g["alpha"]).max()) == 0.0                  # and wrote nothing it could not stand behind
    ctx.ggt_splat_reserve(need)
    g = gpu_splat(ctx, tgt, src, depth)
    assert ctx.ggt_splat_status() == (total, 0)
    assert_same(o, g)
    with pytest.raises(binding.GgtError):
        gpu_splat(ctx, tgt, src, depth, sigma_px=0.0)


def test_splat_c3_shaped_view_with_refine_mask():
    """a rig view of the C3 scene (quarter size) into the held-out target, with the colour image and the Eq. 1 mask that
    ggt_refine_depth's oracle gives for two consecutive frames; then the novel-view mask and Eq. 13"""
    import torch
    from paper_2505_18932_b200 import binding
    wl = synth.workload("C3", scale=0.25)
    tgt = wl.targets(0)[0]
    vi = wl.views_for(tgt)
    ctx = binding.Context()
    o_masks, g_masks = [], []
    for v in vi[:3]:
        d0, c0 = wl.view_inputs(0, v)
        d1, c1 = wl.view_inputs(1, v)
        state, M, _, _ = oracle.refine(c1, c0, d1, d0, theta=8.0 / 255.0)
        o = oracle.splat_forward(tgt, wl.rig[v], state, rgb=c1, mask=M)
        g = gpu_splat(ctx, tgt, wl.rig[v], state, rgb=c1, mask=M)
        assert_same(o, g)
        assert (o["alpha"] > 0.9).mean() > 0.5
        o_masks.append(o["mask"]); g_masks.append(torch.from_numpy(g["mask"]).cuda())
    # Eq. 13 with the splat-and-max mask
    rng = np.random.default_rng(4)
    n = tgt.width * tgt.height
    pd = rng.uniform(0.5, 5, n).astype(np.float32); pd[rng.uniform(size=n) < 0.1] = 0
    pc = rng.uniform(0, 40, n).astype(np.float32); pc[rng.uniform(size=n) < 0.1] = 0
    ow = oracle.temporal_weight_mask(pd, pc, np.maximum.reduce(o_masks).reshape(-1), beta=0.8, eta=15.0)
    gw = torch.empty(n, device="cuda")
    ctx.ggt_temporal_weight_mask(torch.from_numpy(pd).cuda(), torch.from_numpy(pc).cuda(), [m.reshape(-1) for m in g_masks], gw,
                                 beta=0.8, eta=15.0)
    assert np.array_equal(gw.cpu().numpy().view(np.uint32), ow.view(np.uint32))
    assert (ow == 15.0).any() and (ow == 0).any() and ((ow > 0) & (ow < 15)).any()


def test_splat_table4_shape_full_image():
    """PAPER.md Table 4's resolution (1352 x 1014): one rig view into a neighbouring camera, every pixel of
    every output compared (26.7 M list entries)."""
    from paper_2505_18932_b200 import binding
    wl = synth.workload("C3")
    rig = synth.grid_rig(1352, 1014)
    tgt, src = rig[5], rig[6]
    d, rgb = synth.raycast(src, wl.scene, 0.0, want_colour=True)
    d = synth.noisy_depth(d, 7, 1, 0.01, 0.02)
    mask = np.full(d.shape, 0.7, np.float32)
    o = oracle.splat_forward(tgt, src, d, rgb=rgb, mask=mask)
    g = gpu_splat(binding.Context(), tgt, src, d, rgb=rgb, mask=mask)
    assert_same(o, g)
    assert o["count"].max() > 40 and (o["alpha"] == 0).mean() > 0.05

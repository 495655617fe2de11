"""GPU-vs-oracle parity of the paper-style temporal fusion through
the C ABI (-m gpu): ggt_temporal_weight (Eq. 13-14), the *_weighted fusers, and the whole Eq. 3 loop over a video."""
import numpy as np
import pytest

import oracle
from paper_2505_18932_b200 import synth
import helpers

pytestmark = pytest.mark.gpu
TAU = 0.02


def _cuda(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _prev_outputs(tgt, scene, rng, invalid=0.05):
    d = synth.raycast(tgt, scene)[0].astype(np.float32)
    d[rng.uniform(size=d.shape) < invalid] = 0
    acc = rng.uniform(0.0, 20.0, d.shape).astype(np.float32)
    acc[rng.uniform(size=d.shape) < 0.05] = 0
    return d, acc


@pytest.mark.parametrize("n_views,W,H", [(0, 40, 30), (1, 70, 37), (4, 70, 37), (6, 33, 9), (16, 64, 48)])
def test_temporal_weight_parity(n_views, W, H):
    import torch
    from paper_2505_18932_b200 import binding
    wl = synth.workload("C2", scale=0.2)
    rng = np.random.default_rng(100 + n_views)
    rig = synth.grid_rig(W + 13, H + 6)
    prev = synth.camera_from_pose((0.04, -0.03, 0.01), synth.rot_yaw_pitch(0.02, 0.01), 0.8 * W, 0.8 * W, W / 2, H / 2, W, H)
    views = [rig[i] for i in synth.nearest_views(prev, rig, n_views)] if n_views else []
    d, acc = _prev_outputs(prev, wl.scene, rng)
    masks = [rng.uniform(0.6, 1.05, (v.height, v.width)).astype(np.float32) for v in views]
    for beta, eta in ((1.0, 15.0), (0.7, 3.0)):
        ow = oracle.temporal_weight(prev, d, acc, views, masks, beta=beta, eta=eta)
        ctx = binding.Context()
        out = torch.full((H, W), -1.0, dtype=torch.float32, device="cuda")
        ctx.ggt_temporal_weight(prev, _cuda(d), _cuda(acc), views, [_cuda(m) for m in masks], out, beta=beta, eta=eta)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy().view(np.uint32), ow.view(np.uint32))
        assert (ow > 0).any() and (ow == 0).any()


def _extra_view_case(seed=5):
    wl = synth.workload("C2", scale=0.2)
    rng = np.random.default_rng(seed)
    tgt = wl.targets(0)[0]
    vi = wl.views_for(tgt)
    views = [wl.rig[v] for v in vi]
    depths = [wl.view_inputs(0, v)[0] for v in vi]
    prev = synth.camera_from_pose((0.02, 0.01, -0.02), synth.rot_yaw_pitch(-0.01, 0.02), tgt.fx, tgt.fy, tgt.cx, tgt.cy,
                                  tgt.width, tgt.height)
    pd, acc = _prev_outputs(prev, wl.scene, rng)
    w = rng.uniform(0.0, 15.0, pd.shape).astype(np.float32)
    return wl, tgt, views, depths, prev, pd, w


def test_raymarch_weighted_extra_view():
    import torch
    from paper_2505_18932_b200 import binding
    wl, tgt, views, depths, prev, pd, w = _extra_view_case()
    maps = [oracle.weight_map(d) for d in depths] + [oracle.view_record(pd, w)]
    od, oc, on = oracle.raymarch(tgt, views + [prev], maps, 0.5, 5.0, tau=TAU)
    ctx = binding.Context()
    n = tgt.width * tgt.height
    gd, gc = torch.empty(n, device="cuda"), torch.empty(n, device="cuda")
    gn = torch.empty(n, dtype=torch.int32, device="cuda")
    ctx.ggt_raymarch_depth_weighted(tgt, views + [prev], [_cuda(d) for d in depths] + [_cuda(pd)],
                                    [None] * len(views) + [_cuda(w)], 0.5, 5.0, depth=gd, conf=gc, steps=gn, tau=TAU)
    torch.cuda.synchronize()
    assert np.array_equal(gn.cpu().numpy(), on)
    assert np.array_equal(gd.cpu().numpy().view(np.uint32), od.view(np.uint32))
    assert np.array_equal(gc.cpu().numpy().view(np.uint32), oc.view(np.uint32))
    # the extra view matters: without it the result differs
    od0 = oracle.raymarch(tgt, views, maps[:-1], 0.5, 5.0, tau=TAU)[0]
    assert (od0 != od).mean() > 0.2


@pytest.mark.parametrize("dtype_name", ["f32", "f16"])
def test_integrate_weighted_extra_view(dtype_name):
    import torch
    from paper_2505_18932_b200 import binding
    wl, tgt, views, depths, prev, pd, w = _extra_view_case(seed=6)
    maps = [oracle.weight_map(d) for d in depths] + [oracle.view_record(pd, w)]
    tau = oracle.tau_table(wl.z_bins, wl.trunc_bins)
    T, Wt = oracle.integrate(tgt, wl.z_bins, tau, views + [prev], maps, half_storage=dtype_name == "f16")
    od, oc, ob = oracle.extract(wl.z_bins, T, Wt)
    ctx = binding.Context()
    vol = ctx.ggt_volume_bind(tgt.width, tgt.height, wl.z_bins, dtype=binding.GGT_F16 if dtype_name == "f16" else binding.GGT_F32,
                              trunc_bins=wl.trunc_bins)
    vol.ggt_volume_reset()
    ctx.ggt_integrate_weighted(vol, tgt, views + [prev], [_cuda(d) for d in depths] + [_cuda(pd)],
                               [None] * len(views) + [_cuda(w)])
    n = tgt.width * tgt.height
    depth, conf = torch.empty(n, device="cuda"), torch.empty(n, device="cuda")
    bins = torch.empty(n, dtype=torch.int32, device="cuda")
    ctx.ggt_extract_depth(vol, depth, conf, bins)
    st = helpers.compare_frame(dict(rays=None, T=T, W=Wt, depth=od, conf=oc, bins=ob),
                               dict(vol=vol, depth=depth, conf=conf, bins=bins), wl.z_bins, tau)
    helpers.assert_parity(st)
    assert st["T_bitexact"] and st["W_bitexact"]


def test_eq3_video_loop_moving_target():
    """The whole loop of Eq. 3 on the C3-shaped video at 1/4 size over the frames where the target camera changes
    (frame 10): refine with masks -> Eq. 13 weight of D^{t-1} from the PREVIOUS target pose -> weighted raymarch; its
    confidence is the next frame's omega_acc (Eq. 14).  Every frame bit-identical to the oracle."""
    import torch
    from paper_2505_18932_b200 import binding
    wl = synth.workload("C3", scale=0.25)
    op = helpers.OraclePipeline(wl)
    gp = helpers.CudaPipeline(wl)
    ctx = gp.ctx
    o_prev = g_prev = None                       # (camera, depth, conf)
    changed = 0
    for f in range(7, 13):
        tgt = wl.targets(f)[0]
        vi = wl.views_for(tgt)
        views = [wl.rig[v] for v in vi]
        o_ref = [op.refine_view(f, v) for v in vi]                      # (depth, M, pq)
        g_ref = [gp.refine_view(f, v, want_mask=True) for v in vi]
        o_depths = [r[0] for r in o_ref]
        o_masks = [r[1] if r[1] is not None else np.ones_like(r[0]) for r in o_ref]
        g_depths = [r[0] for r in g_ref]
        g_masks = [r[1] for r in g_ref]
        for a, b in zip(o_masks, g_masks):
            assert np.array_equal(a.view(np.uint32), b.cpu().numpy().view(np.uint32))
        maps = [oracle.weight_map(d) for d in o_depths]
        n = tgt.width * tgt.height
        gd, gc = torch.empty(n, device="cuda"), torch.empty(n, device="cuda")
        gn = torch.empty(n, dtype=torch.int32, device="cuda")
        if o_prev is None:
            od, oc, on = oracle.raymarch(tgt, views, maps, 0.5, 5.0, tau=TAU)
            ctx.ggt_raymarch_depth(tgt, views, g_depths, 0.5, 5.0, depth=gd, conf=gc, steps=gn, tau=TAU)
        else:
            pc, pd, pcf = o_prev
            changed += int(not np.array_equal(np.asarray(pc.t), np.asarray(tgt.t)))
            ow = oracle.temporal_weight(pc, pd, pcf, views, o_masks, beta=1.0, eta=15.0)
            rec = oracle.view_record(pd.reshape(pc.height, pc.width), ow)
            od, oc, on = oracle.raymarch(tgt, views + [pc], maps + [rec], 0.5, 5.0, tau=TAU)
            gw = torch.empty((pc.height, pc.width), device="cuda")
            ctx.ggt_temporal_weight(pc, g_prev[1], g_prev[2], views, g_masks, gw, beta=1.0, eta=15.0)
            assert np.array_equal(gw.cpu().numpy().view(np.uint32), ow.view(np.uint32)), "Eq. 13 weight, frame %d" % f
            ctx.ggt_raymarch_depth_weighted(tgt, views + [pc], g_depths + [g_prev[1]], [None] * len(views) + [gw], 0.5, 5.0,
                                            depth=gd, conf=gc, steps=gn, tau=TAU)
        torch.cuda.synchronize()
        assert np.array_equal(gn.cpu().numpy(), on), "frame %d" % f
        assert np.array_equal(gd.cpu().numpy().view(np.uint32), od.view(np.uint32)), "frame %d" % f
        assert np.array_equal(gc.cpu().numpy().view(np.uint32), oc.view(np.uint32)), "frame %d" % f
        o_prev, g_prev = (tgt, od, oc), (tgt, gd, gc)
    assert changed >= 1                                               # the previous pose differed at least once
    plain_conf = oracle.raymarch(tgt, views, maps, 0.5, 5.0, tau=TAU)[1]
    assert (od > 0).mean() > 0.5 and oc.mean() > 1.2 * plain_conf.mean()   # accumulated weight beyond the input views' own


def test_temporal_error_codes():
    import torch
    from paper_2505_18932_b200 import binding
    ctx = binding.Context()
    cam = synth.camera_from_pose((0, 0, 0), np.eye(3), 30, 30, 16.5, 4.5, 33, 9)
    d = torch.full((9, 33), 2.0, device="cuda")
    out = torch.empty((9, 33), device="cuda")
    ctx.ggt_temporal_weight(cam, d, d, [cam], [torch.zeros((9, 33), device="cuda")], out, beta=0.5, eta=15.0)
    torch.cuda.synchronize()
    assert torch.all(out == 1.0)                                      # 0.5 * 2.0 * (1 - 0)
    with pytest.raises(binding.GgtError):
        ctx.ggt_temporal_weight(cam, d, d, [cam], [torch.zeros((9, 33), device="cuda")], out, beta=-1.0)
    with pytest.raises(binding.GgtError):
        ctx.ggt_temporal_weight(cam, d, d, [cam] * 17, [d] * 17, out)

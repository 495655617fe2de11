"""GPU-vs-oracle parity of ggt_raymarch_depth (the paper's own volume-free schedule) through the
C ABI (-m gpu).  Both sides follow the same fp32 operation order (P14), so the sequence of sampled depths
of every ray -- and therefore depth, confidence and the evaluation count -- must be identical bit for bit."""
import numpy as np
import pytest

import oracle
from paper_2505_18932_b200 import synth
import helpers

pytestmark = pytest.mark.gpu
TAU = 0.02


def run_case(tgt, views, depths, z_near, z_far, every=1, seed=1, **kw):
    import torch
    from paper_2505_18932_b200 import binding
    rays = helpers.sample_rays(tgt.width, tgt.height, every, seed)
    okw = dict(kw)
    window = okw.pop("w_window", 7)
    maps = [oracle.weight_map(d, window=window) for d in depths]
    od, oc, on = oracle.raymarch(tgt, views, maps, z_near, z_far, rays=rays, **okw)
    ctx = binding.Context()
    n = tgt.width * tgt.height
    gd = torch.full((n,), -1.0, dtype=torch.float32, device="cuda")
    gc = torch.full((n,), -1.0, dtype=torch.float32, device="cuda")
    gn = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    ctx.ggt_raymarch_depth(tgt, views, [torch.from_numpy(np.ascontiguousarray(d)).cuda() for d in depths], z_near, z_far,
                           depth=gd, conf=gc, steps=gn, **kw)
    torch.cuda.synchronize()
    gd, gc, gn = gd.cpu().numpy(), gc.cpu().numpy(), gn.cpu().numpy()
    if rays is not None:
        gd, gc, gn = gd[rays], gc[rays], gn[rays]
    assert np.array_equal(gn, on), "evaluation counts differ on %d rays" % int((gn != on).sum())
    assert np.array_equal(gd.view(np.uint32), od.view(np.uint32)), "depth differs on %d rays" % int((gd != od).sum())
    assert np.array_equal(gc.view(np.uint32), oc.view(np.uint32))
    # north_star's tolerance, for the record: depth within 1e-4 of the depth range (trivially met when bit-exact)
    assert np.max(np.abs(gd - od)) <= 1e-4 * (z_far - z_near)
    return od, oc, on


def config_inputs(name, scale, frame=0):
    wl = synth.workload(name, scale=scale)
    tgt = wl.targets(frame)[0]
    vi = wl.views_for(tgt)
    return wl, tgt, [wl.rig[v] for v in vi], [wl.view_inputs(frame, v)[0] for v in vi]


def test_raymarch_C1_full():
    wl, tgt, views, depths = config_inputs("C1", 1.0)
    od, oc, on = run_case(tgt, views, depths, 0.5, 4.0, tau=TAU)
    assert (od > 0).mean() > 0.9 and on.max() > 100


def test_raymarch_C2_full_all_rays():
    wl, tgt, views, depths = config_inputs("C2", 1.0)
    od, oc, on = run_case(tgt, views, depths, 0.5, 5.0, tau=TAU)
    assert (od > 0).mean() > 0.5


@pytest.mark.parametrize("name,every", [("C3", 64), ("C4", 64)])
def test_raymarch_full_size_sampled(name, every):
    wl, tgt, views, depths = config_inputs(name, 1.0, frame=1)
    run_case(tgt, views, depths, 0.5, 5.0, every=every, seed=wl.seed, tau=TAU)


def test_raymarch_C5_target_sampled():
    wl, tgt, views, depths = config_inputs("C5", 1.0)      # 2048 x 2048 target, V = 6 views of 1920 x 1080
    run_case(tgt, views, depths, 0.5, 5.0, every=512, seed=wl.seed, tau=TAU)


def _random_rig_case(n_views, W=70, H=37, invalid=False, **kw):
    wl = synth.workload("C2", scale=0.2)
    rig = synth.grid_rig(W + 13, H + 6)
    tgt = synth.camera_from_pose((0.04, -0.03, 0.01), synth.rot_yaw_pitch(0.02, 0.01), 0.8 * W, 0.8 * W, W / 2, H / 2, W, H)
    views = [rig[i] for i in synth.nearest_views(tgt, rig, n_views)]
    depths = []
    for i, c in enumerate(views):
        d = synth.noisy_depth(synth.raycast(c, wl.scene)[0], 11, i, 0.01, 0.03)
        if invalid:
            d[:] = 0
        depths.append(d)
    return run_case(tgt, views, depths, 0.5, 5.0, **kw)


@pytest.mark.parametrize("n_views", [1, 2, 3, 4, 5, 6, 7, 8, 9, 16])
def test_raymarch_view_counts_ragged_sizes(n_views):
    _random_rig_case(n_views, tau=TAU)


def test_raymarch_parameters_and_degenerate_cases():
    od, oc, on = _random_rig_case(4, invalid=True, tau=TAU)          # nothing observed: all misses
    assert np.all(od == 0) and np.all(oc == 0)
    _random_rig_case(4, tau=TAU, max_evals=40)                       # evaluation budget cuts most rays
    _random_rig_case(4, tau=0.05, step_scale=0.5, min_step=3e-3, n_bisect=0)
    _random_rig_case(4, tau=TAU, n_bisect=6, w_window=0)
    _random_rig_case(3, W=33, H=9, tau=TAU)


def test_raymarch_error_codes():
    import torch
    from paper_2505_18932_b200 import binding
    ctx = binding.Context()
    cam = synth.camera_from_pose((0, 0, 0), np.eye(3), 30, 30, 16.5, 4.5, 33, 9)
    d = torch.full((9, 33), 2.0, device="cuda")
    out = torch.empty(33 * 9, device="cuda")
    ctx.ggt_raymarch_depth(cam, [cam], [d], 0.5, 5.0, depth=out)
    torch.cuda.synchronize()
    assert torch.all((out - 2.0).abs() <= 0.8 * TAU / 16 + 1e-6)
    for bad in (dict(z_near=5.0, z_far=0.5), dict(tau=0.0), dict(min_step=0.0), dict(max_evals=0), dict(n_bisect=-1),
                dict(w_window=5)):
        kw = dict(z_near=0.5, z_far=5.0)
        kw.update(bad)
        with pytest.raises(binding.GgtError):
            ctx.ggt_raymarch_depth(cam, [cam], [d], kw.pop("z_near"), kw.pop("z_far"), depth=out, **kw)
    with pytest.raises(binding.GgtError):
        ctx.ggt_raymarch_depth(cam, [], [], 0.5, 5.0, depth=out)
